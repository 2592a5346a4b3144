// mfh_cached.cu -- cached-block streaming matvec: phi^[n] += sum_{m cached} C^[n,m] psi^[m]
// reading HBM-resident blocks (P:177-183 full / partial cache).
//
// HBM-bound: 16 B (c128) / 8 B (c64) of matrix per 4 FMAs.  Cache layout: block-major, each block
// row-major B x B interleaved complex, so a row of a block is one contiguous run of B entries.
// A CTA owns ROWS whole rows of the operator (no atomics, no cross-CTA sums): warp w streams its
// 4 rows with 128-bit non-allocating loads, 4 x 2 independent loads in flight per lane (measured on
// C2: 7.48 TB/s; 2 rows x 4 loads 7.39, 2 x 8 7.33, 1 x 8 7.37, 4 x 4 7.48 at 124 registers); psi^[m]
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
constexpr int CACHED_RPW = 4;                         // rows per warp
constexpr int CACHED_ROWS = CACHED_WARPS * CACHED_RPW;
constexpr int CACHED_U = 2;                           // independent loads per row per lane

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

// --------------------------------------------------------------------------------------------
// k vectors from cached complex128 blocks (coupling scans and the system-bath action in double precision;
// Eq. 12, north_star (c): "reads each V block once for k vectors").  4 k DFMA per 16-byte entry:
// FP64-pipe bound from k = 8 up (k = 16: 64 DFMA per entry = 1 entry/clk/SM = 4.5 TB/s of matrix), HBM bound
// below; there is no FP64 tensor path that would beat the 64 lanes/clk/SM of the CUDA cores, so this is a
// CUDA-core kernel.  A CTA of 128 threads owns 128 rows x one cached block (lane = row, k complex
// accumulators in registers, no reduction); column chunks of 16 entries are staged in shared memory by
// cp.async (16-byte LDGSTS, coalesced 256-byte row runs, double-buffered) in rows padded to 17 entries so
// that the lane = row reads are bank-conflict free; the psi rows of the chunk sit beside them and are read as
// broadcasts.  Output: the partial slot of column block m, as the other k-vector kernels.
// --------------------------------------------------------------------------------------------
constexpr int CM_ROWS = 128, CM_COLS = 16, CM_PAD = CM_COLS + 1;

struct CachedMultiParams {
    int32_t B, n_blk, k, slot_multi;
    int64_t D;
    const int32_t* cache_slot;
    const double2* cache;
    const double2* psi;   // [D][k]
    double2* work;        // [n_slots][D][k]
};

__device__ __forceinline__ void cp_async16(void* dst_smem, const void* src)
{
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"((uint32_t)__cvta_generic_to_shared(dst_smem)), "l"(src)
                 : "memory");
}

// VS = threads per row: each handles KT / VS of the vectors (k = 16 runs two threads per row, which halves the
// accumulator registers per thread and doubles the warps that hide the DFMA and shared-memory latencies).
template <int KT, int VS>
__global__ void __launch_bounds__(CM_ROWS * VS) cached_multi_kernel_c128(const CachedMultiParams P)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    constexpr int TILE = CM_ROWS * CM_PAD;               // entries per stage (padded)
    constexpr int NT = CM_ROWS * VS, KV = KT / VS;
    double2* tiles = reinterpret_cast<double2*>(smem_raw);             // [2][128][17]
    double2* psis = tiles + 2 * TILE;                                  // [2][16][KT]
    const int t = threadIdx.x, row = t & (CM_ROWS - 1), v0 = (t / CM_ROWS) * KV, m = blockIdx.y, k = P.k;
    const int64_t i_base = (int64_t)blockIdx.x * CM_ROWS;
    const int n = (int)(i_base / P.B);
    const int32_t slot = P.cache_slot[n * P.n_blk + m];
    if (slot < 0) return;                                               // generated (or foreign) block
    const double2* blk = P.cache + (size_t)slot * P.B * P.B + (size_t)(i_base - (int64_t)n * P.B) * P.B;
    const double2* psim = P.psi + (size_t)m * P.B * k;
    const int n_chunks = P.B / CM_COLS;

    auto issue = [&](int ch, int st) {
        // 128 rows x 16 entries: thread t copies entry (t & 15) of rows (t >> 4) + (NT / 16) j
        double2* dst = tiles + st * TILE;
        const double2* src = blk + (size_t)ch * CM_COLS + (t & 15);
#pragma unroll
        for (int j = 0; j < CM_ROWS * 16 / NT; ++j) {
            const int r = (t >> 4) + (NT / 16) * j;
            cp_async16(dst + r * CM_PAD + (t & 15), src + (size_t)r * P.B);
        }
        // psi rows of the chunk: 16 x k entries, contiguous in [D][k]
        const double2* ps = psim + (size_t)ch * CM_COLS * k;
        for (int e = t; e < CM_COLS * k; e += NT) cp_async16(psis + st * CM_COLS * KT + (e / k) * KT + (e % k), ps + e);
        asm volatile("cp.async.commit_group;" ::: "memory");
    };

    double2 acc[KV];
#pragma unroll
    for (int v = 0; v < KV; ++v) acc[v] = double2{0.0, 0.0};
    if (k < KT)   // unused vector slots of the staged psi rows stay zero
        for (int e = t; e < 2 * CM_COLS * KT; e += NT) psis[e] = double2{0.0, 0.0};
    __syncthreads();
    issue(0, 0);
    for (int ch = 0; ch < n_chunks; ++ch) {
        const int st = ch & 1;
        if (ch + 1 < n_chunks) {
            issue(ch + 1, st ^ 1);
            asm volatile("cp.async.wait_group 1;" ::: "memory");
        } else {
            asm volatile("cp.async.wait_group 0;" ::: "memory");
        }
        __syncthreads();
        const double2* rowp = tiles + st * TILE + row * CM_PAD;
        const double2* pc = psis + st * CM_COLS * KT + v0;
#pragma unroll 4
        for (int c = 0; c < CM_COLS; ++c) {
            const double2 hv = rowp[c];
#pragma unroll
            for (int v = 0; v < KV; ++v) {
                const double2 p = pc[c * KT + v];
                acc[v].x = fma(hv.x, p.x, acc[v].x);
                acc[v].x = fma(-hv.y, p.y, acc[v].x);
                acc[v].y = fma(hv.x, p.y, acc[v].y);
                acc[v].y = fma(hv.y, p.x, acc[v].y);
            }
        }
        __syncthreads();   // the stage is free for the copy issued in the next iteration
    }
    double2* dst = P.work + ((size_t)(P.slot_multi + m) * P.D + i_base + row) * k + v0;
#pragma unroll
    for (int v = 0; v < KV; ++v)
        if (v0 + v < k) dst[v] = acc[v];
}

bool cached_multi_c128_supported(int dtype, int k, int B) { return dtype == MFH_C128 && k > 1 && k <= MFH_MAX_K && B % CM_ROWS == 0; }

template <int KT, int VS> static int launch_cached_multi_c128_t(mfh_handle h, const void* psi, cudaStream_t st)
{
    const Plan& p = h->plan;
    CachedMultiParams P{p.B, p.n_blk, p.k, p.slot_multi, h->D, h->d_cache_slot, (const double2*)h->d_cache,
                        (const double2*)psi, (double2*)h->d_work};
    const size_t smem = (size_t)(2 * CM_ROWS * CM_PAD + 2 * CM_COLS * KT) * sizeof(double2);
    auto kern = cached_multi_kernel_c128<KT, VS>;
    if (int rc = ensure_dyn_smem(h, kern, (int)smem)) return rc;
    kern<<<dim3((unsigned)(h->D / CM_ROWS), p.n_blk), CM_ROWS * VS, smem, st>>>(P);
    MFH_CUDA_CHECK(cudaGetLastError());
    return MFH_OK;
}

static int launch_cached_multi_c128(mfh_handle h, const void* psi, cudaStream_t st)
{
    const int k = h->plan.k;
    if (k <= 2) return launch_cached_multi_c128_t<2, 1>(h, psi, st);
    if (k <= 4) return launch_cached_multi_c128_t<4, 1>(h, psi, st);
    if (k <= 8) return launch_cached_multi_c128_t<8, 1>(h, psi, st);
    return launch_cached_multi_c128_t<16, 2>(h, psi, st);
}

int launch_cached(mfh_handle h, const void* psi, cudaStream_t st)
{
    const Plan& p = h->plan;
    if (p.n_cached == 0) return MFH_OK;
    if (p.k != 1) {
        if (tc_cached_multi_supported(h->dtype, p.k, p.B)) return launch_cached_multi_tc(h, psi, st);
        if (cached_multi_c128_supported(h->dtype, p.k, p.B)) return launch_cached_multi_c128(h, psi, st);
        set_error("cached blocks with k > 1 need B %% 128 == 0");
        return MFH_ERR_UNSUPPORTED;
    }
    const unsigned grid = (unsigned)(h->D / CACHED_ROWS);
    if (h->dtype == MFH_C128) {
        if (int rc = ensure_dyn_smem(h, cached_kernel_c128, MFH_MAX_B * 16)) return rc;
        CachedParams<double> P{p.B, p.n_blk, p.slot_cache, h->D, h->d_cache_slot,
                               (const double2*)h->d_cache, (const double2*)psi, (double2*)h->d_work};
        cached_kernel_c128<<<grid, 32 * CACHED_WARPS, (size_t)p.B * 16, st>>>(P);
    } else {
        if (int rc = ensure_dyn_smem(h, cached_kernel_c64, MFH_MAX_B * 8)) return rc;
        CachedParams<float> P{p.B, p.n_blk, p.slot_cache, h->D, h->d_cache_slot,
                              (const float2*)h->d_cache, (const float2*)psi, (float2*)h->d_work};
        cached_kernel_c64<<<grid, 32 * CACHED_WARPS, (size_t)p.B * 8, st>>>(P);
    }
    MFH_CUDA_CHECK(cudaGetLastError());
    return MFH_OK;
}

// --------------------------------------------------------------------------------------------
// Hermitian pair cache (cache budget over canonical pairs P:437-446 Eq. 27): block
// C = H^[n,m], n < m, is stored once and every loaded entry is used twice,
//     row side     phi^[n]_a += C_ab psi^[m]_b
//     column side  phi^[m]_b += conj(C_ab) psi^[n]_a
// which halves the HBM bytes per apply.  Work item = a strip of rows of one stored block; a CTA of
// 8 warps pulls items from a device counter.  Warp w owns the column chunks w, w+8, ... (32 U
// 128-bit loads wide), so a lane's columns are fixed while it sweeps the rows of the strip: its
// psi^[m] values and its column accumulators stay in registers and need no reduction at all.  Row
// partials of 4 rows at a time are combined across the 32 lanes by a transposing butterfly
// (24 shuffles per 4 rows instead of 80) and accumulated per (warp,row) in shared memory; at the
// end of the item they are added over the warps in a fixed order.  No atomics; results go to the
// same partial-sum slots as the fused kernel (row side: slot of column block m, column side: slot
// of (row block n, strip)), added in index order by the reduce kernel.
// --------------------------------------------------------------------------------------------
constexpr int PAIR_WARPS = 8;
constexpr int PAIR_THREADS = 32 * PAIR_WARPS;
constexpr int PAIR_RR = 4;   // rows per butterfly
constexpr int PAIR_SR = 256; // rows per sub-strip (shared-memory row partials)

template <typename T> struct PairParams {
    int32_t B, n_blk, n_items, slot_row0;
    int64_t D;
    const ProcItem* items;
    const int32_t* cache_slot;
    const typename Cplx<T>::type* cache;
    const typename Cplx<T>::type* psi;
    typename Cplx<T>::type* work;
    int32_t* counter;
};

template <typename T> struct Vec16;   // one 128-bit load = E entries
template <> struct Vec16<double> {
    static constexpr int E = 1;
    double2 v;
    __device__ __forceinline__ void load(const double2* p) { v = ldg_stream(p); }
    __device__ __forceinline__ double2 get(int) const { return v; }
};
template <> struct Vec16<float> {
    static constexpr int E = 2;
    float4 v;
    __device__ __forceinline__ void load(const float2* p) { v = ldg_stream(reinterpret_cast<const float4*>(p)); }
    __device__ __forceinline__ float2 get(int e) const { return e == 0 ? float2{v.x, v.y} : float2{v.z, v.w}; }
};

// Sum r[0..3] over the 32 lanes; on return every lane holds the total of row 2*bit4 + bit3.
template <typename T> __device__ __forceinline__ T butterfly4(T r0, T r1, T r2, T r3, int lane)
{
    const bool up16 = lane & 16, up8 = lane & 8;
    T k0 = up16 ? r2 : r0, k1 = up16 ? r3 : r1;
    const T s0 = up16 ? r0 : r2, s1 = up16 ? r1 : r3;
    k0 += __shfl_xor_sync(0xffffffffu, s0, 16);
    k1 += __shfl_xor_sync(0xffffffffu, s1, 16);
    T v = up8 ? k1 : k0;
    const T s = up8 ? k0 : k1;
    v += __shfl_xor_sync(0xffffffffu, s, 8);
    v += __shfl_xor_sync(0xffffffffu, v, 4);
    v += __shfl_xor_sync(0xffffffffu, v, 2);
    v += __shfl_xor_sync(0xffffffffu, v, 1);
    return v;
}

template <typename T, int U, int MINB>
__global__ void __launch_bounds__(PAIR_THREADS, MINB) cached_pairs_kernel(const PairParams<T> P)
{
    using CT = typename Cplx<T>::type;
    constexpr int E = Vec16<T>::E, W = PAIR_WARPS, RR = PAIR_RR;
    constexpr int CW = 32 * U * E;                      // columns per warp chunk
    extern __shared__ __align__(16) unsigned char smem_raw[];
    CT* psin = reinterpret_cast<CT*>(smem_raw);         // [nrows]     psi^[n] of the strip
    CT* rowpart = psin + PAIR_SR;                       // [W][nrows]  row partials per warp
    __shared__ int s_item;
    const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
    const int B = P.B, n_chunks = B / CW;

    for (;;) {
        __syncthreads();
        if (tid == 0) s_item = atomicAdd(P.counter, 1);
        __syncthreads();
        const int it = s_item;
        if (it >= P.n_items) break;
        const ProcItem I = P.items[it];
        const bool col_side = (I.col_slot >= 0);
        // rows of the item in sub-strips of at most PAIR_SR rows (shared-memory row partials)
        for (int s0 = 0; s0 < I.nrows; s0 += PAIR_SR) {
            const int nrows = min(PAIR_SR, I.nrows - s0);
            if (s0) __syncthreads();
            for (int a = tid; a < nrows; a += PAIR_THREADS) psin[a] = P.psi[(size_t)I.n * B + I.row0 + s0 + a];
            for (int a = tid; a < W * nrows; a += PAIR_THREADS) rowpart[a] = CT{T(0), T(0)};
            __syncthreads();
            const CT* blk = P.cache + (size_t)P.cache_slot[I.n * P.n_blk + I.m] * B * B + (size_t)(I.row0 + s0) * B;

            for (int ch = w; ch < n_chunks; ch += W) {
                const int c0 = ch * CW + lane * E;          // this lane's columns: c0 + 32 E u + e
                CT pm[U][E], cacc[U][E];
#pragma unroll
                for (int u = 0; u < U; ++u)
#pragma unroll
                    for (int e = 0; e < E; ++e) {
                        pm[u][e] = P.psi[(size_t)I.m * B + c0 + 32 * E * u + e];
                        cacc[u][e] = CT{T(0), T(0)};
                    }
                for (int a = 0; a < nrows; a += RR) {
                    Vec16<T> hv[RR][U];
#pragma unroll
                    for (int r = 0; r < RR; ++r)
#pragma unroll
                        for (int u = 0; u < U; ++u) hv[r][u].load(blk + (size_t)(a + r) * B + c0 + 32 * E * u);
                    T rr_[RR], ri_[RR];
#pragma unroll
                    for (int r = 0; r < RR; ++r) {
                        const CT pn = psin[a + r];
                        T sr = T(0), si = T(0);
#pragma unroll
                        for (int u = 0; u < U; ++u)
#pragma unroll
                            for (int e = 0; e < E; ++e) {
                                const CT hh = hv[r][u].get(e);
                                sr = fma(hh.x, pm[u][e].x, sr);
                                sr = fma(-hh.y, pm[u][e].y, sr);
                                si = fma(hh.x, pm[u][e].y, si);
                                si = fma(hh.y, pm[u][e].x, si);
                                if (col_side) {
                                    cacc[u][e].x = fma(hh.x, pn.x, cacc[u][e].x);     // conj(C_ab) psi_a
                                    cacc[u][e].x = fma(hh.y, pn.y, cacc[u][e].x);
                                    cacc[u][e].y = fma(hh.x, pn.y, cacc[u][e].y);
                                    cacc[u][e].y = fma(-hh.y, pn.x, cacc[u][e].y);
                                }
                            }
                        rr_[r] = sr;
                        ri_[r] = si;
                    }
                    const T tr = butterfly4<T>(rr_[0], rr_[1], rr_[2], rr_[3], lane);
                    const T ti = butterfly4<T>(ri_[0], ri_[1], ri_[2], ri_[3], lane);
                    if ((lane & 7) == 0) {
                        CT& dst = rowpart[w * nrows + a + (lane >> 3)];   // row 2*bit4 + bit3 = lane >> 3
                        dst.x += tr;
                        dst.y += ti;
                    }
                }
                if (col_side) {   // this lane is the only writer of its columns: later sub-strips add in order
                    CT* dst = P.work + (size_t)I.col_slot * P.D + (size_t)I.m * B + c0;
#pragma unroll
                    for (int u = 0; u < U; ++u)
#pragma unroll
                        for (int e = 0; e < E; ++e) {
                            CT v = cacc[u][e];
                            if (s0) {
                                const CT o = dst[32 * E * u + e];
                                v.x += o.x;
                                v.y += o.y;
                            }
                            dst[32 * E * u + e] = v;
                        }
                }
            }
            __syncthreads();
            for (int a = tid; a < nrows; a += PAIR_THREADS) {
                T sr = T(0), si = T(0);
#pragma unroll
                for (int ww = 0; ww < W; ++ww) {
                    const CT v = rowpart[ww * nrows + a];
                    sr += v.x;
                    si += v.y;
                }
                P.work[(size_t)(P.slot_row0 + I.m) * P.D + (size_t)I.n * B + I.row0 + s0 + a] = CT{sr, si};
            }
        }
    }
}

template <typename T, int U, int MINB>
static int launch_pairs_t(mfh_handle h, const void* psi, cudaStream_t st)
{
    using CT = typename Cplx<T>::type;
    const Plan& p = h->plan;
    PairParams<T> P;
    P.B = p.B;
    P.n_blk = p.n_blk;
    P.n_items = (int32_t)p.pair_items.size();
    P.slot_row0 = p.slot_row0;
    P.D = h->D;
    P.items = h->d_pair_items;
    P.cache_slot = h->d_cache_slot;
    P.cache = (const CT*)h->d_cache;
    P.psi = (const CT*)psi;
    P.work = (CT*)h->d_work;
    P.counter = h->d_counter + 1;
    const size_t smem = (size_t)(1 + PAIR_WARPS) * PAIR_SR * sizeof(CT);
    auto kern = cached_pairs_kernel<T, U, MINB>;
    int per_sm = 1;
    MFH_CUDA_CHECK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, PAIR_THREADS, smem));
    if (per_sm < 1) per_sm = 1;
    const int grid = std::min<int>(P.n_items, h->sm_count * per_sm);
    MFH_CUDA_CHECK(cudaMemsetAsync(h->d_counter + 1, 0, sizeof(int32_t), st));
    kern<<<grid, PAIR_THREADS, smem, st>>>(P);
    MFH_CUDA_CHECK(cudaGetLastError());
    return MFH_OK;
}

int launch_cached_pairs(mfh_handle h, const void* psi, cudaStream_t st)
{
    const Plan& p = h->plan;
    if (p.n_cached == 0) return MFH_OK;
    if (p.k != 1) {
        // k vectors (complex64, B % 128 == 0): the tensor-core kernel serves the stored block directly and the mirrored
        // position by a second, transposed read of the same block (mfh_tc.cu)
        if (tc_cached_multi_supported(h->dtype, p.k, p.B)) return launch_cached_multi_tc(h, psi, st);
        set_error("the pair cache with k > 1 needs complex64 and B %% 128 == 0");
        return MFH_ERR_UNSUPPORTED;
    }
    // U 128-bit loads per row per lane x 4 rows in flight; U = 4 at 2 CTAs/SM measured best on C2
    // (7.0 TB/s vs 6.9 for U = 2 at 3 CTAs/SM and 6.6 at 2 CTAs/SM)
    if (h->dtype == MFH_C128) {
        if (p.B % 128 == 0) return launch_pairs_t<double, 4, 2>(h, psi, st);
        if (p.B % 64 == 0) return launch_pairs_t<double, 2, 3>(h, psi, st);
        return launch_pairs_t<double, 1, 4>(h, psi, st);
    }
    return p.B % 128 == 0 ? launch_pairs_t<float, 2, 2>(h, psi, st) : launch_pairs_t<float, 1, 2>(h, psi, st);
}

}  // namespace mfh

// mfh_proc.cu -- generator-side kernels: Philox debug export, block materialisation / cache fill,
// H0 diagonal, and the fused generate-and-apply kernels (single vector with Hermitian reuse,
// k vectors one-sided).  PAPER.md Eq. 7, Eq. 8, Eq. 11.
#include <algorithm>
#include "mfh_internal.cuh"

namespace mfh {

template <typename T> static GenArgs<T> make_gen_args(mfh_handle h);
template <> GenArgs<double> make_gen_args<double>(mfh_handle h)
{
    GenArgs<double> G;
    G.K = make_philox_keys(h->seed);
    G.gc = h->gen_host.gc;
    G.tab_global = h->d_gen_tab;
    G.an = h->analytic;
    return G;
}
template <> GenArgs<float> make_gen_args<float>(mfh_handle h)
{
    GenArgs<float> G;
    G.K = make_philox_keys(h->seed);
    G.gc.neg_k2_ln2 = (float)(-0.6931471805599453 / (double)h->D);
    G.tab_global = nullptr;
    G.an = h->analytic;
    return G;
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
template <typename T, int SRC>
__global__ void __launch_bounds__(256) fill_kernel(const GenArgs<T> G, int32_t B, int32_t n_blk,
                                                   const int32_t* __restrict__ cache_slot,
                                                   int32_t single_n, int32_t single_m, int32_t tiled,
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
    const typename Gen<T>::Tab* tab = stage_gen_table<T>(G);
    __syncthreads();
    for (int32_t a = blockIdx.y; a < B; a += gridDim.y) {
        const uint32_t i = (uint32_t)n * B + a;
        CT* row = out + base + (size_t)a * B;
        for (int32_t b = threadIdx.x; b < B; b += blockDim.x) {
            T hr, hi;
            entry_any<T, SRC>(G, tab, i, (uint32_t)m * B + b, hr, hi);
            CT v;
            v.x = hr;
            v.y = hi;
            if (tiled == 3 && n != m) *reinterpret_cast<CT*>(reinterpret_cast<char*>(out + base) + unit_image_offset(B, a, b)) = v;
            else if (tiled == 1 || tiled == 3) reinterpret_cast<CT*>(reinterpret_cast<T*>(out + base) + tiled_cache_offset(B, a, b))[0] = v;
            else if (tiled == 2) out[base + strip_tile_offset(B, STRIP_PIECE_BYTES / (int)sizeof(CT), a, b)] = v;
            else row[b] = v;
        }
    }
}

template <typename T>
static int launch_fill_t(mfh_handle h, dim3 grid, int32_t B, int32_t n_blk, const int32_t* cache_slot,
                         int32_t n, int32_t m, int32_t tiled, void* out, cudaStream_t st)
{
    using CT = typename Cplx<T>::type;
    if (h->kind == MFH_SRC_ANALYTIC)
        fill_kernel<T, SRC_ANALYTIC><<<grid, 256, 0, st>>>(make_gen_args<T>(h), B, n_blk, cache_slot, n, m,
                                                                            tiled, (CT*)out);
    else
        fill_kernel<T, SRC_SEEDED><<<grid, 256, 0, st>>>(make_gen_args<T>(h), B, n_blk, cache_slot, n, m,
                                                                          tiled, (CT*)out);
    MFH_CUDA_CHECK(cudaGetLastError());
    return MFH_OK;
}

int launch_fill_block(mfh_handle h, int32_t B, int32_t n, int32_t m, void* out, cudaStream_t st)
{
    int rc = ensure_gen_table(h, st);
    if (rc) return rc;
    dim3 grid(1, std::min(B, 1024));
    return h->dtype == MFH_C128 ? launch_fill_t<double>(h, grid, B, 0, nullptr, n, m, 0, out, st)
                                : launch_fill_t<float>(h, grid, B, 0, nullptr, n, m, 0, out, st);
}

int launch_fill_cache(mfh_handle h, cudaStream_t st)
{
    const Plan& p = h->plan;
    if (p.n_cached == 0) return MFH_OK;
    int rc = ensure_gen_table(h, st);
    if (rc) return rc;
    dim3 grid(p.n_blk * p.n_blk, std::min(p.B, 64));
    // layouts: 0 row-major blocks, 1 the 16 KB tiles of complex64 k-vector plans, 2 the strip tiles of partial plans,
    // 3 a k-vector pair cache: unit images for the off-diagonal blocks, 16 KB tiles for the diagonal ones
    const int strip = p.strip_tiled ? 2 : 0;
    return h->dtype == MFH_C128
               ? launch_fill_t<double>(h, grid, p.B, p.n_blk, h->d_cache_slot, 0, 0, strip, h->d_cache, st)
               : launch_fill_t<float>(h, grid, p.B, p.n_blk, h->d_cache_slot, 0, 0, p.k > 1 ? (p.pair_units ? 3 : 1) : strip, h->d_cache, st);
}

// External block (Eq. 10) -> cache slot: a plain copy for row-major caches, a re-layout for the tiled cache
// of complex64 k-vector plans (mfh_internal.cuh tiled_cache_offset).
__global__ void __launch_bounds__(256) retile_kernel(int32_t B, int32_t units, const float2* __restrict__ src, float2* __restrict__ dst)
{
    for (int64_t e = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; e < (int64_t)B * B; e += (int64_t)gridDim.x * blockDim.x) {
        const int a = (int)(e / B), b = (int)(e % B);
        if (units) *reinterpret_cast<float2*>(reinterpret_cast<char*>(dst) + unit_image_offset(B, a, b)) = src[e];
        else reinterpret_cast<float2*>(reinterpret_cast<float*>(dst) + tiled_cache_offset(B, a, b))[0] = src[e];
    }
}

// (n, m): the block's position -- an off-diagonal block of a k-vector pair cache is stored as unit images
int launch_store_block_at(mfh_handle h, int32_t slot, int32_t n, int32_t m, const void* src_dev, cudaStream_t st)
{
    const Plan& p = h->plan;
    const size_t cb = complex_bytes(h->dtype), bytes = (size_t)p.B * p.B * cb;
    char* dst = (char*)h->d_cache + (size_t)slot * bytes;
    if (h->dtype == MFH_C64 && p.k > 1) {
        retile_kernel<<<std::min(p.B * p.B / 256, 148 * 8), 256, 0, st>>>(p.B, (p.pair_units && n != m) ? 1 : 0, (const float2*)src_dev, (float2*)dst);
        MFH_CUDA_CHECK(cudaGetLastError());
    } else {
        MFH_CUDA_CHECK(cudaMemcpyAsync(dst, src_dev, bytes, cudaMemcpyDeviceToDevice, st));
    }
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
// (n,m) for a one-sided item).  The CTA walks the strip in row tiles of TR = 32 R rows: lane l
// owns the R rows l, l+32, ... of the tile (psi_i and the row accumulators stay in registers for
// the whole tile), warp w owns the 32-column sub-tiles w, w+W, ... of the block, so every column
// belongs to exactly one warp: no atomics, and no barrier inside a tile.  In a sub-tile, at step s
// lane l handles column (l+s) mod 32 of its R rows: each entry H_ij (i<j) is generated once in
// registers and used twice,
//     row side     phi_i += H_ij psi_j              (accumulator stays in lane l)
//     column side  phi_j += conj(H_ij) psi_i        (accumulator rotates lane l+1 -> l each step)
// so after 32 steps lane l holds the complete column-l sum of the sub-tile, which the owning warp
// adds to the CTA's shared column array.  Row sums are combined across the W warps through shared
// memory in a fixed order at the end of each tile.  Results go to partial-sum slots that the
// reduce kernel adds in index order (deterministic, repeatable bit for bit).
// --------------------------------------------------------------------------------------------
constexpr int PROC_WARPS = 8;
constexpr int PROC_THREADS = 32 * PROC_WARPS;

template <typename T> struct ProcParams {
    GenArgs<T> G;
    int32_t B, n_blk, n_items, slot_row0;
    int64_t D;
    const ProcItem* items;
    const typename Cplx<T>::type* psi;
    typename Cplx<T>::type* work;   // [n_slots][D]
    int32_t* counter;
    // fused tail (small procedural plans: one launch per apply).  done[b] counts the finished contributions to block
    // row b; the CTA that delivers the last one adds the block row's partial slots in list order and writes phi.
    int32_t* done;                  // nullptr: the reduce kernel runs after this one
    int32_t* fin;                   // CTAs that have left the item loop (the last one resets the item counter)
    const int32_t* expected;        // [n_blk] contributions per block row
    const int32_t* slot_list;       // [n_blk][n_slots + 1]
    int32_t n_slots;
    const T* h0;                    // H0 diagonal or nullptr
    typename Cplx<T>::type* phi;
    double lambda;
};

// phi^[b] = h0 (.) psi^[b] + lambda * sum over the valid slots of block row b, in ascending slot order (the order of
// reduce_kernel's plain path): partial sums written by other CTAs are read through L2 (ld.global.cg).
template <typename T>
__device__ __forceinline__ void reduce_block_row(const ProcParams<T>& P, int b)
{
    using CT = typename Cplx<T>::type;
    const int32_t* list = P.slot_list + (size_t)b * (P.n_slots + 1);
    const int cnt = list[0] & SLOT_COUNT_MASK;
    for (int a = threadIdx.x; a < P.B; a += PROC_THREADS) {
        const size_t i = (size_t)b * P.B + a;
        double sr = 0.0, si = 0.0;
        int t = 0;
        for (; t + 8 <= cnt; t += 8) {   // eight independent loads in flight, added in list order
            CT x[8];
#pragma unroll
            for (int u = 0; u < 8; ++u) x[u] = __ldcg(P.work + (size_t)list[1 + t + u] * P.D + i);
#pragma unroll
            for (int u = 0; u < 8; ++u) {
                sr += (double)x[u].x;
                si += (double)x[u].y;
            }
        }
        for (; t < cnt; ++t) {
            const CT x = __ldcg(P.work + (size_t)list[1 + t] * P.D + i);
            sr += (double)x.x;
            si += (double)x.y;
        }
        double outr = P.lambda * sr, outi = P.lambda * si;
        if (P.h0) {
            const CT p = P.psi[i];
            const double d = (double)P.h0[i];
            outr = fma(d, (double)p.x, outr);
            outi = fma(d, (double)p.y, outi);
        }
        CT o;
        o.x = (T)outr;
        o.y = (T)outi;
        P.phi[i] = o;
    }
}

// The item loop of one CTA: runs until the device counter is exhausted.
template <typename T, int R, int SRC = SRC_SEEDED>
__device__ __forceinline__ void proc_items(const ProcParams<T>& P, unsigned char* smem_raw)
{
    using CT = typename Cplx<T>::type;
    constexpr int W = PROC_WARPS, TR = 32 * R;
    const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
    const int B = P.B;
    const typename Gen<T>::Tab* tab = stage_gen_table<T>(P.G);
    CT* colsum = reinterpret_cast<CT*>(smem_raw);                      // [B]     column-side sums of the item
    CT* rowred = colsum + B;                                           // [W][TR] row sums of the tile per warp
    CT* psiw = rowred + W * TR + w * 32;                               // [32]    psi of the warp's sub-tile
    __shared__ int s_item, s_red[2];
    const int n_ct = B / 32;

    for (;;) {
        __syncthreads();
        if (tid == 0) s_item = atomicAdd(P.counter, 1);
        __syncthreads();
        const int it = s_item;
        if (it >= P.n_items) break;
        const ProcItem I = P.items[it];
        const bool one_sided_item = (I.kind == PAIR_ONE_SIDED);
        const bool diag_item = (I.kind == PAIR_DIAG);
        for (int c = tid; c < B; c += PROC_THREADS) colsum[c] = CT{T(0), T(0)};
        __syncthreads();

        for (int rt = I.row0 / TR; rt < (I.row0 + I.nrows) / TR; ++rt) {
            const uint32_t i0 = (uint32_t)I.n * B + rt * TR + lane;
            CT psi_i[R];
            T accr[R], acci[R];
#pragma unroll
            for (int r = 0; r < R; ++r) {
                psi_i[r] = P.psi[i0 + 32 * r];
                accr[r] = acci[r] = T(0);
            }
            // diagonal block: sub-tiles left of the tile's diagonal square are covered by transposes
            const int cs_first = diag_item ? rt * R : 0;
            for (int cs = cs_first + w; cs < n_ct; cs += W) {
                const uint32_t j0 = (uint32_t)I.m * B + cs * 32;
                __syncwarp();
                psiw[lane] = P.psi[j0 + lane];
                __syncwarp();
                if (one_sided_item || (diag_item && cs < (rt + 1) * R)) {
#pragma unroll 1
                    for (int s = 0; s < 32; ++s) {
                        const int c = (lane + s) & 31;
                        const CT p = psiw[c];
#pragma unroll
                        for (int r = 0; r < R; ++r) {
                            T hr, hi;
                            entry_any<T, SRC>(P.G, tab, i0 + 32 * r, j0 + c, hr, hi);
                            accr[r] = fma(hr, p.x, accr[r]);
                            accr[r] = fma(-hi, p.y, accr[r]);
                            acci[r] = fma(hr, p.y, acci[r]);
                            acci[r] = fma(hi, p.x, acci[r]);
                        }
                    }
                } else {
                    T cr = T(0), ci = T(0);
#pragma unroll 1
                    for (int s = 0; s < 32; ++s) {
                        const int c = (lane + s) & 31;
                        const CT p = psiw[c];
#pragma unroll
                        for (int r = 0; r < R; ++r) {
                            T hr, hi;
                            entry_upper<T, SRC>(P.G, tab, i0 + 32 * r, j0 + c, hr, hi);
                            accr[r] = fma(hr, p.x, accr[r]);
                            accr[r] = fma(-hi, p.y, accr[r]);
                            acci[r] = fma(hr, p.y, acci[r]);
                            acci[r] = fma(hi, p.x, acci[r]);
                            cr = fma(hr, psi_i[r].x, cr);     // conj(H_ij) psi_i
                            cr = fma(hi, psi_i[r].y, cr);
                            ci = fma(hr, psi_i[r].y, ci);
                            ci = fma(-hi, psi_i[r].x, ci);
                        }
                        cr = __shfl_sync(0xffffffffu, cr, (lane + 1) & 31);
                        ci = __shfl_sync(0xffffffffu, ci, (lane + 1) & 31);
                    }
                    CT& dst = colsum[cs * 32 + lane];   // this warp is the only writer of these columns
                    dst.x += cr;
                    dst.y += ci;
                }
            }
#pragma unroll
            for (int r = 0; r < R; ++r) rowred[w * TR + lane + 32 * r] = CT{accr[r], acci[r]};
            __syncthreads();
            if (tid < TR) {
                T sr = T(0), si = T(0);
#pragma unroll
                for (int ww = 0; ww < W; ++ww) {
                    const CT v = rowred[ww * TR + tid];
                    sr += v.x;
                    si += v.y;
                }
                P.work[(size_t)(P.slot_row0 + I.m) * P.D + (size_t)I.n * B + rt * TR + tid] = CT{sr, si};
            }
            __syncthreads();
        }
        if (I.col_slot >= 0) {
            CT* dst = P.work + (size_t)I.col_slot * P.D + (size_t)I.m * B;
            for (int c = tid; c < B; c += PROC_THREADS) dst[c] = colsum[c];
        }
        if (P.done) {
            __threadfence();                 // this thread's partial sums are visible device-wide ...
            __syncthreads();                 // ... before thread 0 announces the item
            if (tid == 0) {
                int r0 = -1, r1 = -1;
                if (atomicAdd(&P.done[I.n], 1) == P.expected[I.n] - 1) r0 = I.n;
                if (I.col_slot >= 0 && atomicAdd(&P.done[I.m], 1) == P.expected[I.m] - 1) r1 = I.m;
                if (r0 >= 0) P.done[r0] = 0;   // last contribution of this launch: leave the counter clean for the next
                if (r1 >= 0) P.done[r1] = 0;
                s_red[0] = r0;
                s_red[1] = r1;
                __threadfence();
            }
            __syncthreads();
            for (int q = 0; q < 2; ++q)
                if (s_red[q] >= 0) reduce_block_row<T>(P, s_red[q]);
        }
    }
    if (P.done && tid == 0 && atomicAdd(P.fin, 1) == (int)gridDim.x - 1) {
        *P.counter = 0;                      // every CTA has left the item loop: self-cleaning, no memset launch
        *P.fin = 0;
    }
}

template <typename T, int R, int SRC = SRC_SEEDED>
__global__ void __launch_bounds__(PROC_THREADS, 2) proc_single_kernel(const ProcParams<T> P)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    proc_items<T, R, SRC>(P, smem_raw);
}

// --------------------------------------------------------------------------------------------
// Partial-cache mode, overlapped (Eq. 33: T = max of the cached and the generated part
// instead of their sum).  The cached part loads the memory pipe, the generated part the ALU
// pipes, but two kernels that each fill the SMs run back to back.  So both parts run in ONE
// persistent kernel with two CTAs per SM: CTAs of the first wave prefer fused generate-and-apply
// items, CTAs of the second wave prefer cached row strips, and whoever exhausts its own queue
// takes work from the other (two device counters).  A cached strip is 32 whole operator rows
// (4 per warp, 4 x 4 independent 128-bit streaming loads per lane = 64 KB in flight per CTA)
// over all cached blocks of the block row, psi^[m] staged in shared memory: the loop of
// cached_kernel_c128 made persistent.  Same partial-sum slots and the same fixed-order reduce.
// --------------------------------------------------------------------------------------------
template <typename T> struct StripParams {
    int32_t B, n_blk, slot_cache, n_strips;
    int64_t D;
    const int32_t* cache_slot;
    const typename Cplx<T>::type* cache;
    const typename Cplx<T>::type* psi;
    typename Cplx<T>::type* work;
    int32_t* counter;
};

// Streaming role.  A strip is STRIP_ROWS = 8 whole operator rows over all cached blocks of the block row.  The bytes
// are moved by the TMA engine, not by load instructions: STRIP_WS warps per CTA each run their OWN two-stage ring --
// a stage is one 8 KB tile of the strip-tiled cache layout (8 row pieces of 1 KB, contiguous: ONE bulk copy) plus the
// matching 1 KB of psi^[m] -- and multiply what they loaded themselves: no CTA-wide barrier, no hand-over between
// warps.  Measured on B200: bulk copies issued by one thread are serviced one after the other
// (~0.27 us each whatever their size up to 32 KB), copies of different warps overlap; a register-staged loop tops
// out near 56 GB/s per SM, a CTA-wide ring with one issuing thread near 30 GB/s per CTA, per-warp rings reach the
// ~125 GB/s an SM's 64 B/clk port allows -- which is what lets FEW SMs pull most of the HBM bandwidth while the
// others generate.  Lane = 16-byte unit of a row piece; 8 complex row accumulators per lane, summed over the lanes by
// shuffles at the end of the strip, one warp per strip: no atomics, fixed summation order.
constexpr int STRIP_ROWS = 8;                   // rows per strip (and per tile)
constexpr int STRIP_PIECE = STRIP_PIECE_BYTES;   // bytes of one row piece (and of the psi piece)
constexpr int STRIP_TILE = STRIP_ROWS * STRIP_PIECE;
constexpr int STRIP_STAGE = STRIP_TILE + STRIP_PIECE;
constexpr int STRIP_WS = 4;                     // streaming warps per CTA (one per scheduler)
constexpr int STRIP_SMEM = STRIP_WS * 2 * STRIP_STAGE;

__device__ __forceinline__ uint32_t sm_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void sm_mbar_wait(uint64_t* bar, uint32_t parity)
{
    uint32_t done;
    do {
        asm volatile(
            "{\n\t"
            ".reg .pred p;\n\t"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
            "selp.u32 %0, 1, 0, p;\n\t"
            "}\n"
            : "=r"(done)
            : "r"(sm_u32(bar)), "r"(parity)
            : "memory");
    } while (!done);
}
__device__ __forceinline__ void bulk_load(void* dst_smem, const void* src, uint32_t bytes, uint64_t* bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(sm_u32(dst_smem)),
                 "l"(src), "r"(bytes), "r"(sm_u32(bar))
                 : "memory");
}

// acc += h * p for the 16-byte unit: one complex128 entry, or two complex64 entries
__device__ __forceinline__ void unit_fma(const double2& h, const double2& p, double& ar, double& ai)
{
    ar = fma(h.x, p.x, ar);
    ar = fma(-h.y, p.y, ar);
    ai = fma(h.x, p.y, ai);
    ai = fma(h.y, p.x, ai);
}
__device__ __forceinline__ void unit_fma(const float4& h, const float4& p, float& ar, float& ai)
{
    ar = fmaf(h.x, p.x, ar);
    ar = fmaf(-h.y, p.y, ar);
    ai = fmaf(h.x, p.y, ai);
    ai = fmaf(h.y, p.x, ai);
    ar = fmaf(h.z, p.z, ar);
    ar = fmaf(-h.w, p.w, ar);
    ai = fmaf(h.z, p.w, ai);
    ai = fmaf(h.w, p.z, ai);
}
template <typename T> struct Unit16;
template <> struct Unit16<double> { using type = double2; };
template <> struct Unit16<float> { using type = float4; };

template <typename T>
__device__ __forceinline__ void cached_strips(const StripParams<T>& S, unsigned char* smem_raw)
{
    using CT = typename Cplx<T>::type;
    using U16 = typename Unit16<T>::type;
    constexpr int COLS = STRIP_PIECE / (int)sizeof(CT);     // columns per piece
    constexpr int UPL = STRIP_PIECE / 16 / 32;              // 16-byte units per lane and row piece
    __shared__ __align__(8) uint64_t full[STRIP_WS][2];
    const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
    if (w < STRIP_WS) {
        const int B = S.B, chunks = B / COLS;
        unsigned char* ring = smem_raw + (size_t)w * 2 * STRIP_STAGE;
        if (lane == 0) {
            asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(sm_u32(&full[w][0])), "r"(1) : "memory");
            asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(sm_u32(&full[w][1])), "r"(1) : "memory");
            asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        }
        __syncwarp();
        uint32_t g = 0;                       // tiles this warp has consumed so far (stage = g & 1, parity = (g >> 1) & 1)
        for (;;) {
            int it = 0;
            if (lane == 0) it = atomicAdd(S.counter, 1);
            it = __shfl_sync(0xffffffffu, it, 0);
            if (it >= S.n_strips) break;
            const int64_t row0 = (int64_t)it * STRIP_ROWS;
            const int n = (int)(row0 / B), a0 = (int)(row0 % B);
            const int32_t* slots = S.cache_slot + (size_t)n * S.n_blk;
            // tile sequence of the strip: cached blocks in ascending m (fixed summation order), column chunks inside
            int m_next = 0, ch_next = 0;      // next tile to ISSUE
            int32_t slot_next = -1;
            auto advance_block = [&]() {      // move (m_next, slot_next) to the next cached block, or past the end
                while (m_next < S.n_blk && (slot_next = slots[m_next]) < 0) ++m_next;
            };
            advance_block();
            auto issue = [&](uint32_t gi) {   // issue the next tile of the sequence into stage gi & 1; false at the end
                if (m_next >= S.n_blk) return false;
                if (lane == 0) {
                    unsigned char* dst = ring + (size_t)(gi & 1u) * STRIP_STAGE;
                    uint64_t* bar = &full[w][gi & 1u];
                    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // the stage was read by generic loads
                    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(sm_u32(bar)), "r"(STRIP_STAGE) : "memory");
                    bulk_load(dst, S.cache + (size_t)slot_next * B * B + strip_tile_offset(B, COLS, a0, ch_next * COLS), STRIP_TILE, bar);
                    bulk_load(dst + STRIP_TILE, S.psi + (size_t)m_next * B + (size_t)ch_next * COLS, STRIP_PIECE, bar);
                }
                if (++ch_next == chunks) {
                    ch_next = 0;
                    ++m_next;
                    advance_block();
                }
                return true;
            };
            T ar[STRIP_ROWS], ai[STRIP_ROWS];
#pragma unroll
            for (int r = 0; r < STRIP_ROWS; ++r) ar[r] = ai[r] = T(0);
            int in_flight = 0;
            if (issue(g)) ++in_flight;
            if (issue(g + 1)) ++in_flight;
            while (in_flight > 0) {
                const uint32_t st = g & 1u;
                sm_mbar_wait(&full[w][st], (g >> 1) & 1u);
                const U16* tile = reinterpret_cast<const U16*>(ring + (size_t)st * STRIP_STAGE);
                const U16* psip = tile + STRIP_TILE / 16;
                U16 pv[UPL];
#pragma unroll
                for (int q = 0; q < UPL; ++q) pv[q] = psip[lane + 32 * q];
#pragma unroll
                for (int r = 0; r < STRIP_ROWS; ++r) {
                    U16 hv[UPL];
#pragma unroll
                    for (int q = 0; q < UPL; ++q) hv[q] = tile[r * (STRIP_PIECE / 16) + lane + 32 * q];
#pragma unroll
                    for (int q = 0; q < UPL; ++q) unit_fma(hv[q], pv[q], ar[r], ai[r]);
                }
                __syncwarp();                 // every lane has read the stage: it may be refilled
                --in_flight;
                if (issue(g + 2)) ++in_flight;
                ++g;
            }
#pragma unroll
            for (int r = 0; r < STRIP_ROWS; ++r) {
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) {
                    ar[r] += __shfl_xor_sync(0xffffffffu, ar[r], o);
                    ai[r] += __shfl_xor_sync(0xffffffffu, ai[r], o);
                }
                if (lane == r) S.work[(size_t)S.slot_cache * S.D + row0 + r] = CT{ar[r], ai[r]};
            }
        }
    }
    __syncthreads();                          // the idle warps wait here; the shared memory is free for the next role
}

// SM-partitioned roles (Eq. 33): the CTAs of `stream_sms` SMs -- spread evenly over the SM ids -- stream cached strips,
// the CTAs of the other SMs generate; whoever exhausts its own queue takes work from the other.  Both CTAs of an SM
// have the same role, so a streaming warp never shares an SM with generator warps except in the tail.
__device__ __forceinline__ bool sm_streams(int stream_sms, int n_sm)
{
    uint32_t smid;
    asm("mov.u32 %0, %%smid;" : "=r"(smid));
    smid %= (uint32_t)n_sm;
    return ((smid + 1) * (uint32_t)stream_sms) / (uint32_t)n_sm != (smid * (uint32_t)stream_sms) / (uint32_t)n_sm;
}

template <typename T, int R>
__global__ void __launch_bounds__(PROC_THREADS, 2)
partial_overlap_kernel(const ProcParams<T> P, const StripParams<T> S, int stream_sms, int n_sm)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    if (!sm_streams(stream_sms, n_sm)) {
        proc_items<T, R>(P, smem_raw);
        cached_strips<T>(S, smem_raw);
    } else {
        cached_strips<T>(S, smem_raw);
        proc_items<T, R>(P, smem_raw);
    }
}

template <typename T, int R>
static int launch_proc_single_t(mfh_handle h, const void* psi, void* phi, double lambda, cudaStream_t st)
{
    using CT = typename Cplx<T>::type;
    const Plan& p = h->plan;
    ProcParams<T> P;
    const bool fused = h->fused_tail && phi != nullptr;
    P.done = fused ? h->d_counter + 3 : nullptr;
    P.fin = h->d_counter + 2;
    P.expected = h->d_expected;
    P.slot_list = h->d_slot_list;
    P.n_slots = std::max(p.n_slots, 1);
    P.h0 = (const T*)h->d_h0;
    P.phi = (CT*)phi;
    P.lambda = lambda;
    P.G = make_gen_args<T>(h);
    P.B = p.B;
    P.n_blk = p.n_blk;
    P.n_items = (int32_t)p.items.size();
    P.slot_row0 = p.slot_row0;
    P.D = h->D;
    P.items = h->d_items;
    P.psi = (const CT*)psi;
    P.work = (CT*)h->d_work;
    P.counter = h->d_counter;
    auto smem_for = [](int B) {
        return (size_t)(B + PROC_WARPS * 32 * R + PROC_WARPS * 32) * sizeof(CT);   // + the static generator table
    };
    const size_t smem = smem_for(p.B);
    const bool analytic = (h->kind == MFH_SRC_ANALYTIC);
    auto kern = analytic ? proc_single_kernel<T, R, SRC_ANALYTIC> : proc_single_kernel<T, R, SRC_SEEDED>;
    if (int rc = ensure_dyn_smem(h, kern, (int)smem_for(MFH_MAX_B))) return rc;
    int per_sm = 1;
    MFH_CUDA_CHECK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, PROC_THREADS, smem));
    if (per_sm < 1) per_sm = 1;
    const int grid = std::min<int>(P.n_items, h->sm_count * per_sm);
    if (!fused) MFH_CUDA_CHECK(cudaMemsetAsync(h->d_counter, 0, sizeof(int32_t), st));   // the fused tail resets it itself
    kern<<<grid, PROC_THREADS, smem, st>>>(P);
    MFH_CUDA_CHECK(cudaGetLastError());
    return MFH_OK;
}

// phi != nullptr on a handle with fused_tail: the kernel also reduces (one launch per apply) and the caller skips
// launch_reduce.
int launch_proc_single(mfh_handle h, const void* psi, void* phi, double lambda, cudaStream_t st)
{
    if (h->plan.items.empty()) return MFH_OK;
    const bool f64 = (h->dtype == MFH_C128);
    switch (h->plan.R) {
    case 4: return f64 ? launch_proc_single_t<double, 4>(h, psi, phi, lambda, st) : launch_proc_single_t<float, 4>(h, psi, phi, lambda, st);
    case 2: return f64 ? launch_proc_single_t<double, 2>(h, psi, phi, lambda, st) : launch_proc_single_t<float, 2>(h, psi, phi, lambda, st);
    case 1: return f64 ? launch_proc_single_t<double, 1>(h, psi, phi, lambda, st) : launch_proc_single_t<float, 1>(h, psi, phi, lambda, st);
    }
    set_error("unsupported rows per lane %d", h->plan.R);
    return MFH_ERR_INVALID_ARG;
}

bool partial_overlap_supported(mfh_handle h)
{
    const Plan& p = h->plan;
    const int cols = STRIP_PIECE / (int)complex_bytes(h->dtype);   // a row piece must not cross a block
    return h->kind != MFH_SRC_ANALYTIC && p.k == 1 && !p.pairs && p.n_cached > 0 && !p.items.empty() && p.B % cols == 0;
}

template <typename T, int R> static int launch_partial_overlap_t(mfh_handle h, const void* psi, cudaStream_t st)
{
    using CT = typename Cplx<T>::type;
    const Plan& p = h->plan;
    ProcParams<T> P;
    P.G = make_gen_args<T>(h);
    P.B = p.B;
    P.n_blk = p.n_blk;
    P.n_items = (int32_t)p.items.size();
    P.slot_row0 = p.slot_row0;
    P.D = h->D;
    P.items = h->d_items;
    P.psi = (const CT*)psi;
    P.work = (CT*)h->d_work;
    P.counter = h->d_counter;
    P.done = nullptr;
    P.fin = nullptr;
    StripParams<T> S;
    S.B = p.B;
    S.n_blk = p.n_blk;
    S.slot_cache = p.slot_cache;
    S.n_strips = (int32_t)(h->D / STRIP_ROWS);
    S.D = h->D;
    S.cache_slot = h->d_cache_slot;
    S.cache = (const CT*)h->d_cache;
    S.psi = (const CT*)psi;
    S.work = (CT*)h->d_work;
    S.counter = h->d_counter + 1;
    // dynamic shared memory: the generator's arrays or the streaming ring, whichever is larger, with two CTAs per SM
    const size_t gen_smem = (size_t)(p.B + PROC_WARPS * 32 * R + PROC_WARPS * 32) * sizeof(CT);   // + the static generator table
    auto kern = partial_overlap_kernel<T, R>;
    if (int rc = ensure_dyn_smem(h, kern, 96 * 1024)) return rc;
    const size_t smem = std::max(gen_smem, (size_t)STRIP_SMEM);
    int per_sm = 0;
    MFH_CUDA_CHECK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, PROC_THREADS, smem));
    if (per_sm < 1) {
        set_error("partial plan: the fused kernel does not fit an SM (B = %d)", p.B);
        return MFH_ERR_UNSUPPORTED;
    }
    const int grid = h->sm_count * per_sm;
    MFH_CUDA_CHECK(cudaMemsetAsync(h->d_counter, 0, 2 * sizeof(int32_t), st));
    const int stream_sms = p.stream_sms > 0 ? std::min(p.stream_sms, h->sm_count - 1) : h->sm_count / 3;
    kern<<<grid, PROC_THREADS, smem, st>>>(P, S, stream_sms, h->sm_count);
    MFH_CUDA_CHECK(cudaGetLastError());
    return MFH_OK;
}

int launch_partial_overlap(mfh_handle h, const void* psi, cudaStream_t st)
{
    const bool f64 = (h->dtype == MFH_C128);
    switch (h->plan.R) {
    case 4: return f64 ? launch_partial_overlap_t<double, 4>(h, psi, st) : launch_partial_overlap_t<float, 4>(h, psi, st);
    case 2: return f64 ? launch_partial_overlap_t<double, 2>(h, psi, st) : launch_partial_overlap_t<float, 2>(h, psi, st);
    case 1: return f64 ? launch_partial_overlap_t<double, 1>(h, psi, st) : launch_partial_overlap_t<float, 1>(h, psi, st);
    }
    set_error("unsupported rows per lane %d", h->plan.R);
    return MFH_ERR_INVALID_ARG;
}

// --------------------------------------------------------------------------------------------
// Fused generate-and-apply, k vectors (coupling scans, Eq. 12): every V entry is
// generated ONCE per apply and multiplied into all k columns.  One-sided: lane = row, a CTA owns
// 32W rows x one uncached column block m (blockIdx.y), the psi rows of a column chunk are staged
// in shared memory and read as broadcasts; k accumulators per lane stay in registers and go to
// the partial slot of column block m (added in index order by the reduce kernel).
// --------------------------------------------------------------------------------------------
template <typename T> struct MultiParams {
    GenArgs<T> G;
    int32_t B, n_blk, k, slot_multi;
    int64_t D;
    const int32_t* cache_slot;
    const typename Cplx<T>::type* psi;   // [D][k]
    typename Cplx<T>::type* work;        // [n_slots][D][k]
};

template <typename T, int KT, int W, int SRC = SRC_SEEDED>
__global__ void __launch_bounds__(32 * W) proc_multi_kernel(const MultiParams<T> P)
{
    using CT = typename Cplx<T>::type;
    constexpr int CH = 32;                         // columns per staged chunk
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const typename Gen<T>::Tab* tab = stage_gen_table<T>(P.G);
    CT(*psis)[KT] = reinterpret_cast<CT(*)[KT]>(smem_raw);                       // [CH][KT]
    const int tid = threadIdx.x;
    const uint32_t i = blockIdx.x * (32 * W) + tid;
    const int n = (int)(i / (uint32_t)P.B);
    const int k = P.k;
    CT acc[KT];
#pragma unroll
    for (int v = 0; v < KT; ++v) acc[v] = CT{T(0), T(0)};

    const int m = blockIdx.y;
    if (P.cache_slot[n * P.n_blk + m] != -1) return;   // cached block: the streaming kernel covers it
    {
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
                entry_any<T, SRC>(P.G, tab, i, j0 + c, hr, hi);
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
    CT* dst = P.work + ((size_t)(P.slot_multi + m) * P.D + i) * k;
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
    P.G = make_gen_args<T>(h);
    P.B = p.B;
    P.n_blk = p.n_blk;
    P.k = p.k;
    P.slot_multi = p.slot_multi;
    P.D = h->D;
    P.cache_slot = h->d_cache_slot;
    P.psi = (const CT*)psi;
    P.work = (CT*)h->d_work;
    const size_t smem = 32 * KT * sizeof(CT);
    // 32W rows per CTA must divide B; prefer 128-row CTAs, fall back to one warp.
    const bool analytic = (h->kind == MFH_SRC_ANALYTIC);
    if (p.B % 128 == 0) {
        const dim3 grid((unsigned)(h->D / 128), p.n_blk);
        if (analytic) proc_multi_kernel<T, KT, 4, SRC_ANALYTIC><<<grid, 128, smem, st>>>(P);
        else proc_multi_kernel<T, KT, 4, SRC_SEEDED><<<grid, 128, smem, st>>>(P);
    } else {
        const dim3 grid((unsigned)(h->D / 32), p.n_blk);
        if (analytic) proc_multi_kernel<T, KT, 1, SRC_ANALYTIC><<<grid, 32, smem, st>>>(P);
        else proc_multi_kernel<T, KT, 1, SRC_SEEDED><<<grid, 32, smem, st>>>(P);
    }
    MFH_CUDA_CHECK(cudaGetLastError());
    return MFH_OK;
}

int launch_proc_multi(mfh_handle h, const void* psi, cudaStream_t st)
{
    // complex64, B % 128 == 0: tensor-core kernel (mfh_tc.cu)
    if (tc_multi_supported(h)) return launch_proc_multi_tc(h, psi, st);
    const int k = h->plan.k;
    const bool f64 = (h->dtype == MFH_C128);
    if (k <= 2) return f64 ? launch_proc_multi_t<double, 2>(h, psi, st) : launch_proc_multi_t<float, 2>(h, psi, st);
    if (k <= 4) return f64 ? launch_proc_multi_t<double, 4>(h, psi, st) : launch_proc_multi_t<float, 4>(h, psi, st);
    if (k <= 8) return f64 ? launch_proc_multi_t<double, 8>(h, psi, st) : launch_proc_multi_t<float, 8>(h, psi, st);
    return f64 ? launch_proc_multi_t<double, 16>(h, psi, st) : launch_proc_multi_t<float, 16>(h, psi, st);
}

}  // namespace mfh

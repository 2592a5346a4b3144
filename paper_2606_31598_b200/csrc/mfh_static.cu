// mfh_static.cu -- mfh_apply_static: phi = lambda V(seed) psi without any allocation (include/mfh.h).
//
// For callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that forbid
// it): no handle, no plan, no cudaMalloc / cudaFree / allocating library routine anywhere on this path.  It is a variant
// of the generate-and-apply kernel for one complex128 vector (Eq. 4-5; entries as BASELINE.json configs[0]),
// one-sided (every entry generated where it is used, no Hermitian reuse), whose scratch -- the generator table and the
// partial sums per column chunk that the fixed-order reduction adds, the same two things the handle path keeps in
// cudaMalloc'ed buffers -- lives in ONE file-scope device array of fixed size:
//     [0, 32 KB)            generator table of the last D applied on this device (mfh_gen.cuh GenTabD, 20.3 KB)
//     [32 KB, 32 KB + 4 MB) partial sums [chunk c < 16][row i < D] complex128, D <= MFH_STATIC_MAX_D = 16384
// Every GPU that loads the library holds these 4.03 MB until the process exits.
// The array keeps the last call's contents and EVERY call on a device shares it: calls that overlap on the GPU (two
// streams, two threads) race on it -- the caller serialises them.  Nothing has to start at zero: every partial sum the
// reduction reads is written by the same call's first kernel (all 16 chunk slots of all D rows; chunks beyond the
// matrix get an explicit zero), and the table is re-uploaded whenever D differs from the table's.
#include <algorithm>
#include <mutex>
#include "mfh_internal.cuh"

namespace mfh {

constexpr int64_t ST_MAX_D = MFH_STATIC_MAX_D;
constexpr int ST_CHUNKS = 16;                      // column chunks = partial sums per row
constexpr int ST_ROWS = 128;                       // rows per CTA (thread = row)
constexpr size_t ST_TAB_BYTES = 32768;             // room for GenTabD
constexpr size_t ST_PART_BYTES = (size_t)ST_CHUNKS * ST_MAX_D * sizeof(double2);
static_assert(sizeof(GenTabD) <= ST_TAB_BYTES, "generator table does not fit its slot of the static scratch");

// In HOST code this name is a host-side stand-in, not a device address: the address comes from cudaGetSymbolAddress.
static __device__ __align__(256) unsigned char g_static_scratch[ST_TAB_BYTES + ST_PART_BYTES];

// partial[c][i] = sum over the columns j of chunk c of V_ij psi_j  (row tile blockIdx.x, chunk blockIdx.y)
__global__ void __launch_bounds__(ST_ROWS) static_partial_kernel(const GenArgs<double> G, int64_t D, int32_t W,
                                                                 const double2* __restrict__ psi, double2* __restrict__ partial)
{
    __shared__ double2 s_psi[ST_ROWS];
    const Gen<double>::Tab* tab = stage_gen_table<double>(G);
    const int tid = threadIdx.x;
    const uint32_t i = blockIdx.x * ST_ROWS + tid;
    const int64_t j_begin = (int64_t)blockIdx.y * W, j_end = min(D, j_begin + W);
    double sr = 0.0, si = 0.0;
    for (int64_t j0 = j_begin; j0 < j_end; j0 += ST_ROWS) {   // W and D are multiples of ST_ROWS
        __syncthreads();                                      // table staged / previous piece consumed
        s_psi[tid] = psi[j0 + tid];
        __syncthreads();
#pragma unroll 2
        for (int jj = 0; jj < ST_ROWS; ++jj) {
            double hr, hi;
            entry_any<double>(G, tab, i, (uint32_t)(j0 + jj), hr, hi);
            const double2 x = s_psi[jj];
            sr = fma(hr, x.x, sr);
            sr = fma(-hi, x.y, sr);
            si = fma(hr, x.y, si);
            si = fma(hi, x.x, si);
        }
    }
    partial[(size_t)blockIdx.y * D + i] = make_double2(sr, si);   // an empty chunk writes its zero
}

// phi_i = lambda * (partial[0][i] + partial[1][i] + ... ) in index order
__global__ void __launch_bounds__(256) static_reduce_kernel(int64_t D, double lambda, const double2* __restrict__ partial,
                                                            double2* __restrict__ phi)
{
    const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (i >= D) return;
    double sr = 0.0, si = 0.0;
#pragma unroll
    for (int c = 0; c < ST_CHUNKS; ++c) {
        const double2 x = partial[(size_t)c * D + i];
        sr += x.x;
        si += x.y;
    }
    phi[i] = make_double2(lambda * sr, lambda * si);
}

// Per device: the scratch's device address (cudaGetSymbolAddress, once, with that device current) and the D whose
// generator table sits in the scratch.
struct StaticDev {
    unsigned char* ptr = nullptr;
    int64_t table_D = 0;
};
constexpr int ST_MAX_DEVICES = 64;
static StaticDev g_static_dev[ST_MAX_DEVICES];
static GenHostD g_static_host;   // host copy of the table being uploaded (guarded by the mutex)
static int64_t g_static_host_D = 0;
static std::mutex g_static_mutex;

}  // namespace mfh

using namespace mfh;

MFH_API int mfh_apply_static(int64_t D, uint64_t seed, double lambda, const void* psi_dev, void* phi_dev, void* stream)
{
    if (!psi_dev || !phi_dev || psi_dev == phi_dev) {
        set_error("mfh_apply_static: NULL or aliased pointer");
        return MFH_ERR_INVALID_ARG;
    }
    if (D > ST_MAX_D) {
        set_error("mfh_apply_static: D = %lld exceeds the static scratch (MFH_STATIC_MAX_D = %lld); use mfh_create / mfh_plan / mfh_apply",
                  (long long)D, (long long)ST_MAX_D);
        return MFH_ERR_INVALID_ARG;
    }
    if (D < ST_ROWS || D % ST_ROWS != 0) {
        set_error("mfh_apply_static: D = %lld must be a multiple of %d (and at least %d)", (long long)D, ST_ROWS, ST_ROWS);
        return MFH_ERR_INVALID_ARG;
    }
    cudaStream_t st = (cudaStream_t)stream;
    int dev = -1;
    MFH_CUDA_CHECK(cudaGetDevice(&dev));
    if (dev < 0 || dev >= ST_MAX_DEVICES) {
        set_error("mfh_apply_static: device ordinal %d not supported (at most %d devices)", dev, ST_MAX_DEVICES);
        return MFH_ERR_UNSUPPORTED;
    }
    std::lock_guard<std::mutex> lock(g_static_mutex);
    StaticDev& S = g_static_dev[dev];
    if (!S.ptr) {   // set-up, once per device, with that device current
        unsigned char* p = nullptr;
        MFH_CUDA_CHECK(cudaGetSymbolAddress((void**)&p, g_static_scratch));
        S.ptr = p;
        S.table_D = 0;
    }
    if (g_static_host_D != D) {
        make_gen_table(D, g_static_host);
        g_static_host_D = D;
    }
    if (S.table_D != D) {
        // stream-ordered after the previous call's kernels; the pageable source is consumed before the call returns
        MFH_CUDA_CHECK(cudaMemcpyAsync(S.ptr, &g_static_host.tab, sizeof(GenTabD), cudaMemcpyHostToDevice, st));
        S.table_D = D;
    }
    GenArgs<double> G;
    G.K = make_philox_keys(seed);
    G.gc = g_static_host.gc;
    G.tab_global = reinterpret_cast<const GenTabD*>(S.ptr);
    G.an = AnalyticArgs{0, 0, 1, 0, 0, 0, 0};
    double2* partial = reinterpret_cast<double2*>(S.ptr + ST_TAB_BYTES);
    const int tiles = (int)(D / ST_ROWS);
    const int32_t W = ST_ROWS * ((tiles + ST_CHUNKS - 1) / ST_CHUNKS);   // columns per chunk: ceil(tiles / 16) row tiles wide
    static_partial_kernel<<<dim3((unsigned)tiles, ST_CHUNKS), ST_ROWS, 0, st>>>(G, D, W, (const double2*)psi_dev, partial);
    MFH_CUDA_CHECK(cudaGetLastError());
    static_reduce_kernel<<<(unsigned)((D + 255) / 256), 256, 0, st>>>(D, lambda, partial, (double2*)phi_dev);
    MFH_CUDA_CHECK(cudaGetLastError());
    return MFH_OK;
}

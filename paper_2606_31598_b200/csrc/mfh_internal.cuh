// mfh_internal.cuh -- handle, plan tables and launcher prototypes shared by the .cu files.
#pragma once
#include <cstdint>
#include <cstdio>
#include <string>
#include <utility>
#include <vector>
#include <cuda_runtime.h>

#include "mfh.h"
#include "mfh_gen.cuh"

namespace mfh {

template <typename T> struct Cplx;
template <> struct Cplx<double> { using type = double2; };
template <> struct Cplx<float> { using type = float2; };

// Block-pair roles in the procedural kernel (host table N_blk x N_blk, row n, column m).
enum : uint8_t {
    PAIR_NONE = 0,      // not generated from (n,m): cached, or covered by the mirrored pair (m,n)
    PAIR_TWO_SIDED = 1, // n < m, both (n,m) and (m,n) uncached: generate once, use for both
    PAIR_ONE_SIDED = 2, // generate (n,m) for phi^[n] only
    PAIR_DIAG = 3       // n == m: upper sub-tiles two-sided, diagonal sub-tiles one-sided
};

// One work item of the single-vector procedural kernel: a strip of rows of block n times all
// columns of block m.
struct ProcItem {
    int32_t n, m;       // block pair
    int32_t row0;       // first row of the strip inside block n
    int32_t nrows;      // strip height (multiple of the macro tile)
    int32_t kind;       // PAIR_*
    int32_t col_slot;   // partial slot receiving the column-side sums (-1: none)
};

// Tiled cache layout of k-vector plans (complex64): element (a, b) of a B x B block, in floats from the
// block start.  Tiles of 128 rows x 32 floats (16 complex columns) are contiguous 16 KB runs, ordered
// column tile fastest inside a row tile; inside a tile row r holds 8 chunks of 16 bytes, chunk c stored
// at position c ^ (r & 7) (the 128-byte swizzle the tensor-core kernel reads conflict-free).
__host__ __device__ inline size_t tiled_cache_offset(int B, int a, int b)
{
    const int rt = a >> 7, r = a & 127, kt = b >> 4, c = (b & 15) >> 1;
    return ((size_t)rt * (B >> 4) + kt) * 4096 + (size_t)r * 32 + (size_t)((c ^ (r & 7)) << 2) + (size_t)((b & 1) << 1);
}

// Unit-image layout of the off-diagonal blocks of a complex64 k-vector PAIR cache (two-sided cached kernel,
// mfh_tc.cu): element (a, b) of a B x B block, in BYTES from the block start.  A unit = 128 rows x 32 columns = 32 KB
// contiguous (one bulk copy), units ordered column range fastest inside a 128-row strip.  Inside a unit the image is
// the K-major, 128-byte-swizzled shared-memory B operand of the column side (row = block column, K = (block row,
// re/im)): [(r % 64) / 16] 8 KB, [r / 64] 4 KB, [c / 8] 1 KB, [c % 8] 128 B, 16-byte chunk ((r % 16) / 2) ^ (c % 8),
// [r % 2] 8 B -- exactly what the generator threads of pairs_tc_kernel write for a generated unit.
__host__ __device__ inline size_t unit_image_offset(int B, int a, int b)
{
    const int strip = a >> 7, r = a & 127, u = b >> 5, c = b & 31;
    return ((size_t)strip * (B >> 5) + u) * 32768 + (size_t)((r & 63) >> 4) * 8192 + (size_t)(r >> 6) * 4096 + (size_t)(c >> 3) * 1024 +
           (size_t)(c & 7) * 128 + (size_t)((((r & 15) >> 1) ^ (c & 7)) << 4) + (size_t)(r & 1) * 8;
}

// Strip-tiled cache layout of one-vector PARTIAL plans (the streaming role of partial_overlap_kernel, mfh_proc.cu):
// element (a, b) of a B x B block, in complex elements from the block start.  A tile is 8 rows x `cols` columns
// (cols = STRIP_PIECE_BYTES of complex: 64 complex128 / 128 complex64), 8 KB contiguous, tiles ordered column chunk
// fastest inside an 8-row strip -- so a strip's pass over a block is one contiguous run and every stage of a
// streaming warp's ring is ONE bulk copy.
constexpr int STRIP_PIECE_BYTES = 1024;
__host__ __device__ inline size_t strip_tile_offset(int B, int cols, int a, int b)
{
    return ((size_t)(a >> 3) * (B / cols) + (size_t)(b / cols)) * (size_t)(8 * cols) + (size_t)(a & 7) * cols + (size_t)(b % cols);
}

struct Plan {
    int32_t mode = 0;          // MFH_MODE_* actually committed
    int32_t B = 0, n_blk = 0, k = 0;
    int32_t Q = 1;             // row strips per block in the procedural kernel
    int32_t R = 4;             // rows per lane in the procedural kernel (row tile = 32*R rows)
    int32_t stream_sms = 0;    // partial plans: SMs whose CTAs stream cached blocks while the others generate (Eq. 33)
    bool pairs = false;        // Hermitian pair cache: store block (n,m), n <= m, use it for both sides
    bool strip_tiled = false;  // cached blocks stored in the strip-tiled layout (partial plans run by partial_overlap_kernel)
    bool pair_units = false;   // complex64 k-vector pair cache: off-diagonal stored blocks in the unit-image layout, served
                               // for both sides from ONE read by cached_pairs_tc_kernel
    int64_t n_cached = 0;      // stored blocks
    int64_t covered_blocks = 0;   // block positions (n,m) served from the cache
    int32_t cached_per_row = 0;
    int32_t n_slots = 0;       // partial vectors in the workspace
    int32_t slot_cache = -1, slot_row0 = -1, slot_col0 = -1, slot_multi = -1;
    int32_t slot_mcol0 = -1;   // k-vector two-sided generator (mfh_tc.cu): column-side slots, one per (row block, 128-row strip)
    bool allow_tc_pairs = true;   // caller: the column-side slots of the two-sided k-vector kernels fit the budget
    bool gen_two_sided = true;    // caller: the source is seeded (the two-sided tensor-core GENERATOR is the Philox path)
    size_t cache_bytes = 0, work_bytes = 0;
    int32_t part_rank = 0, part_world = 1, part_scheme = 0;   // mfh_set_partition
    int64_t owned_blocks = 0;     // block positions this rank is responsible for (n_blk^2 on one GPU)
    int32_t row_first = 0, row_count = 0;   // block rows of phi this rank writes
    std::vector<uint8_t> own;          // [n_blk*n_blk] 1 = position owned by this rank
    std::vector<int32_t> cache_slot;   // [n_blk*n_blk] cached block index, -1 generated, -2 served by the mirrored pair, -3 not owned
    std::vector<uint8_t> pair_kind;    // [n_blk*n_blk]
    std::vector<ProcItem> items;       // fused generate-and-apply kernel
    std::vector<ProcItem> pair_items;  // cached pair kernel (pairs mode)
    std::vector<int32_t> tc_pairs;     // k-vector two-sided generator: (row block, column block) of every pair it serves
    std::vector<uint8_t> tc_skip;      // [n_blk*n_blk] 1 = position served by a two-sided kernel (the one-sided kernels skip it)
    std::vector<int32_t> tc_left;      // generated positions the two-sided generator leaves to the one-sided kernel: (row block, column block)
    std::vector<int32_t> ct_left;      // cached positions the two-sided cached kernel leaves to cached_multi_tc_kernel
    std::vector<int32_t> tc_cpairs;    // two-sided cached kernel: (row block, column block, cache slot) of every stored pair
    std::vector<uint8_t> slot_valid;   // [n_blk][n_slots]
    std::string json;
};

}  // namespace mfh

struct mfh_handle_s {
    int64_t D = 0;
    int32_t B_req = 0;
    uint64_t seed = 0, seed_h0 = 0;
    int32_t kind = 0, dtype = 0;
    double lambda = 1.0;
    mfh::AnalyticArgs analytic = {0, 0, 1, 0, 0, 0, 0};          // mfh_set_source_params (MFH_SRC_ANALYTIC)
    bool analytic_set = false;
    std::vector<uint8_t> ext_set;                                 // MFH_SRC_EXTERNAL: per cache slot, block supplied
    int64_t ext_missing = 0;                                      // stored blocks not supplied yet
    int32_t part_rank = 0, part_world = 1, part_scheme = 0;   // mfh_set_partition
    mfh_exchange_fn exchange = nullptr;                       // mfh_set_exchange
    void* exchange_user = nullptr;
    bool planned = false;
    mfh::Plan plan;
    // device resources (library-owned)
    void* d_cache = nullptr;
    void* d_work = nullptr;         // partial slots: [n_slots][D][k] complex
    void* d_h0 = nullptr;           // D reals (DIAG_PLUS_GUE)
    int32_t* d_cache_slot = nullptr;
    mfh::ProcItem* d_items = nullptr;
    mfh::ProcItem* d_pair_items = nullptr;
    int32_t* d_tc_pairs = nullptr;    // plan.tc_pairs
    uint8_t* d_tc_skip = nullptr;     // plan.tc_skip
    int32_t* d_tc_cpairs = nullptr;   // plan.tc_cpairs
    int32_t* d_tc_left = nullptr;     // plan.tc_left
    int32_t* d_ct_left = nullptr;     // plan.ct_left
    int32_t* d_slot_list = nullptr;   // [n_blk][n_slots+1]: count | flags, then the valid slots in ascending order
    double* d_lambdas = nullptr;    // MFH_MAX_K doubles, refreshed by every apply
    int32_t* d_counter = nullptr;   // dynamic work counters: [0] procedural kernel, [1] pair kernel, [2] CTAs finished,
                                    // [3 .. 3 + n_blk) finished contributions per block row (fused tail)
    int32_t* d_expected = nullptr;  // [n_blk] contributions the fused tail waits for per block row
    bool fused_tail = false;        // small procedural k = 1 plans: the fused kernel also reduces (one launch per apply)
    void* d_cheb = nullptr;         // 3 vectors of Chebyshev scratch
    void* d_io = nullptr;           // psi/phi staging of mfh_apply_host
    void* d_lanczos = nullptr;      // 3 Lanczos vectors + alpha/beta/norm scalars + reduction partials
    mfh::GenHostD gen_host;         // generator table + constants for this D (host copy)
    mfh::GenTabD* d_gen_tab = nullptr;   // device copy (c128 only), kept until mfh_destroy
    bool gen_ready = false;
    int sm_count = 148;
    int device = -1;                // the CUDA device the plan lives on (set by mfh_plan)
    // kernels whose cudaFuncAttributeMaxDynamicSharedMemorySize has been raised on `device` for this handle: the
    // attribute is per device, so it is remembered per handle, not per process
    std::vector<std::pair<const void*, int>> smem_attr;
    void* d_stage = nullptr;        // mfh_set_block: one reusable B x B staging block (tiled caches)
    std::vector<std::pair<void*, size_t>> guarded;   // (allocation base, user bytes) of every guarded plan buffer
    std::vector<cudaEvent_t> timing_events;   // mfh_timing_begin: 4 events per armed apply
    int32_t timing_n = 0, timing_pos = 0;
};

namespace mfh {

// flags in the count word of a block row's slot list (reduce kernel)
constexpr int32_t SLOT_SKIP_ROW = 1 << 30;   // MFH_PART_ROWS: block row not owned, phi left untouched
constexpr int32_t SLOT_NO_H0 = 1 << 29;      // MFH_PART_PAIRS: diagonal block on another rank, no h0 (.) psi term
constexpr int32_t SLOT_COUNT_MASK = (1 << 29) - 1;

void set_error(const char* fmt, ...);
size_t complex_bytes(int dtype);

#define MFH_CUDA_CHECK(expr)                                                                   \
    do {                                                                                       \
        cudaError_t _e = (expr);                                                               \
        if (_e != cudaSuccess) {                                                               \
            mfh::set_error("%s failed: %s (%s:%d)", #expr, cudaGetErrorString(_e), __FILE__,   \
                           __LINE__);                                                          \
            return MFH_ERR_CUDA;                                                               \
        }                                                                                      \
    } while (0)

// Raise the dynamic shared-memory limit of `kernel` to `bytes` on the handle's device (once per handle and kernel).
template <typename K> inline int ensure_dyn_smem(mfh_handle h, K kernel, int bytes)
{
    const void* f = reinterpret_cast<const void*>(kernel);
    for (const auto& e : h->smem_attr)
        if (e.first == f && e.second >= bytes) return MFH_OK;
    MFH_CUDA_CHECK(cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes));
    h->smem_attr.push_back({f, bytes});
    return MFH_OK;
}

int ensure_gen_table(mfh_handle h, cudaStream_t st);   // mfh_api.cu: build + upload once per handle

// ---- launchers (mfh_proc.cu, mfh_cached.cu, mfh_vec.cu) ----
int launch_philox_debug(uint64_t seed, uint32_t stream_id, const uint32_t* i, const uint32_t* j,
                        int64_t n, uint32_t* words, cudaStream_t st);
int launch_fill_block(mfh_handle h, int32_t B, int32_t n, int32_t m, void* out, cudaStream_t st);
int launch_fill_cache(mfh_handle h, cudaStream_t st);
int launch_h0(mfh_handle h, void* out, cudaStream_t st);
int launch_proc_single(mfh_handle h, const void* psi, void* phi, double lambda, cudaStream_t st);
bool partial_overlap_supported(mfh_handle h);
int launch_partial_overlap(mfh_handle h, const void* psi, cudaStream_t st);   // cached + generated in one kernel
int launch_proc_multi(mfh_handle h, const void* psi, cudaStream_t st);
bool tc_multi_supported(mfh_handle h);                                   // mfh_tc.cu
int launch_proc_multi_tc(mfh_handle h, const void* psi, cudaStream_t st);
bool tc_pairs_supported(int dtype, int k, int B);        // two-sided tensor-core generator
bool tc_cached_multi_supported(int dtype, int k, int B);
bool cached_multi_c128_supported(int dtype, int k, int B);               // mfh_cached.cu
int launch_cached_multi_tc(mfh_handle h, const void* psi, cudaStream_t st);
int launch_cached_pairs_tc(mfh_handle h, const void* psi, cudaStream_t st);
int launch_store_block_at(mfh_handle h, int32_t slot, int32_t n, int32_t m, const void* src_dev, cudaStream_t st);
int launch_cached(mfh_handle h, const void* psi, cudaStream_t st);
int launch_cached_pairs(mfh_handle h, const void* psi, cudaStream_t st);
int launch_reduce(mfh_handle h, const void* psi, void* phi, const double* lambdas_host, cudaStream_t st);
int launch_cheb_first(mfh_handle h, const void* psi, void* q_prev, void* acc, double j0,
                      cudaStream_t st);
int launch_cheb_step(mfh_handle h, const void* hq, const void* q, void* prev_dst, void* acc, double c,
                     double inv_r, int first, double coef_re, double coef_im, cudaStream_t st);
int launch_cheb_final(mfh_handle h, const void* acc, void* out, double ph_re, double ph_im,
                      cudaStream_t st);
int launch_lz_dot(mfh_handle h, const void* x, const void* y, double* partial, double* dst, int take_sqrt, cudaStream_t st);
int launch_lz_update(mfh_handle h, void* w, const void* v, const void* v_prev, const double* alpha, const double* beta_prev,
                     double* partial, double* beta_dst, cudaStream_t st);
int launch_lz_scale(mfh_handle h, const void* src, void* dst, const double* scale, cudaStream_t st);
int lz_partial_doubles();

}  // namespace mfh

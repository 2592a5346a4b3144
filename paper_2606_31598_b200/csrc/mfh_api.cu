// mfh_api.cu -- the C ABI of include/mfh.h: argument checking, plan commit, apply dispatch,
// the Chebyshev driver and the test exports.  Every step of the path runs in the kernels of
// mfh_proc.cu / mfh_cached.cu / mfh_vec.cu; this file only marshals.
#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstring>
#include "mfh_internal.cuh"
#include "mfh_plan.h"

namespace mfh {

static thread_local char g_err[1024] = "";

void set_error(const char* fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof g_err, fmt, ap);
    va_end(ap);
}

size_t complex_bytes(int dtype) { return dtype == MFH_C128 ? 16 : 8; }

static void copy_json(const std::string& s, char* out, size_t cap)
{
    if (!out || cap == 0) return;
    const size_t n = std::min(s.size(), cap - 1);
    memcpy(out, s.data(), n);
    out[n] = 0;
}

static bool valid_B(int64_t D, int32_t B)
{
    return B >= MFH_MIN_B && B <= MFH_MAX_B && B % MFH_MIN_B == 0 && D % B == 0;
}

// Every library-owned device buffer of a plan is allocated with a guard band of GUARD_BYTES on both sides, filled
// with GUARD_BYTE.  mfh_debug_selfcheck counts the guard bytes that no longer hold the pattern: an out-of-bounds
// WRITE of any kernel into or next to these buffers shows up there (compute-sanitizer is closed on this pool).
static const size_t GUARD_BYTES = 4096;
static const unsigned char GUARD_BYTE = 0xA5;

static cudaError_t guarded_malloc(mfh_handle h, void** user, size_t bytes)
{
    char* base = nullptr;
    cudaError_t e = cudaMalloc(&base, bytes + 2 * GUARD_BYTES);
    if (e != cudaSuccess) return e;
    e = cudaMemset(base, GUARD_BYTE, GUARD_BYTES);
    if (e == cudaSuccess) e = cudaMemset(base + GUARD_BYTES + bytes, GUARD_BYTE, GUARD_BYTES);
    if (e != cudaSuccess) { cudaFree(base); return e; }
    *user = base + GUARD_BYTES;
    h->guarded.push_back({base, bytes});
    return cudaSuccess;
}

static int free_plan_resources(mfh_handle h)
{
    void** ptrs[] = {&h->d_cache, &h->d_work, &h->d_h0, (void**)&h->d_cache_slot, (void**)&h->d_items,
                     (void**)&h->d_pair_items, (void**)&h->d_tc_pairs, (void**)&h->d_tc_skip, (void**)&h->d_tc_cpairs, (void**)&h->d_tc_left, (void**)&h->d_ct_left,
                     (void**)&h->d_slot_list, (void**)&h->d_counter, (void**)&h->d_expected, &h->d_cheb, &h->d_io, &h->d_lanczos, &h->d_stage};
    for (void** p : ptrs) *p = nullptr;
    for (auto& g : h->guarded) cudaFree(g.first);
    h->guarded.clear();
    h->planned = false;
    return MFH_OK;
}

int ensure_gen_table(mfh_handle h, cudaStream_t st)
{
    if (h->gen_ready) return MFH_OK;
    make_gen_table(h->D, h->gen_host);
    if (h->dtype == MFH_C128) {
        if (!h->d_gen_tab) MFH_CUDA_CHECK(cudaMalloc(&h->d_gen_tab, sizeof(GenTabD)));
        MFH_CUDA_CHECK(cudaMemcpyAsync(h->d_gen_tab, &h->gen_host.tab, sizeof(GenTabD), cudaMemcpyHostToDevice, st));
        MFH_CUDA_CHECK(cudaStreamSynchronize(st));   // gen_host is pageable: make the copy complete
    }
    h->gen_ready = true;
    return MFH_OK;
}

// Scratch of the chained drivers (library-owned, allocated by mfh_plan): Chebyshev cur, prev, acc, Hq + the ping-pong
// vector of mfh_chebyshev_steps; Lanczos v, v_prev, w + alpha[4096], beta[4096], 8 scalars and the reduction partials.
static size_t cheb_scratch_bytes(int64_t D, int dtype, int k) { return (size_t)5 * D * k * complex_bytes(dtype); }
static size_t lanczos_scratch_bytes(int64_t D, int dtype)
{
    return (size_t)3 * D * complex_bytes(dtype) + (2 * 4096 + 8 + (size_t)lz_partial_doubles()) * sizeof(double);
}

// Largest D whose procedural k = 1 plans fold the reduce into the fused kernel (one launch per apply).  The reduce of
// a block row is done by the ONE CTA that delivers its last contribution, so it pays off only while a block row's
// partial sums are small: measured at C1 (D = 4096, 72 partial slots, 590 KB per block row) the single launch is
// 2-3 us SLOWER than kernel + reduce kernel (59.0 against 55.4 us per apply replayed from a graph: the apply is bound
// by the one-item-per-CTA generator wave, not by launches), so the tail is kept for D <= 2048 only.
static const int64_t kFusedTailMaxD = 2048;

// Allocate and upload everything plan `p` needs, then fill the cache.
static int commit_plan(mfh_handle h, const Plan& p, cudaStream_t st)
{
    free_plan_resources(h);
    h->plan = p;
    h->plan.strip_tiled = partial_overlap_supported(h);   // the streaming role reads 16 KB tiles (mfh_proc.cu)
    const Plan& q = h->plan;
    const size_t cb = complex_bytes(h->dtype);
    cudaError_t e;
    if (q.cache_bytes) {
        e = guarded_malloc(h, (void**)&h->d_cache, q.cache_bytes);
        if (e != cudaSuccess) {
            cudaGetLastError();
            set_error("cache allocation of %zu bytes failed: %s", q.cache_bytes, cudaGetErrorString(e));
            free_plan_resources(h);
            return MFH_ERR_OUT_OF_MEMORY;
        }
    }
    e = guarded_malloc(h, (void**)&h->d_work, q.work_bytes);
    if (e != cudaSuccess) {
        cudaGetLastError();
        set_error("workspace allocation of %zu bytes failed: %s", q.work_bytes, cudaGetErrorString(e));
        free_plan_resources(h);
        return MFH_ERR_OUT_OF_MEMORY;
    }
    MFH_CUDA_CHECK(guarded_malloc(h, (void**)&h->d_cache_slot, q.cache_slot.size() * sizeof(int32_t)));
    MFH_CUDA_CHECK(cudaMemcpyAsync(h->d_cache_slot, q.cache_slot.data(), q.cache_slot.size() * sizeof(int32_t),
                                   cudaMemcpyHostToDevice, st));
    if (!q.items.empty()) {
        MFH_CUDA_CHECK(guarded_malloc(h, (void**)&h->d_items, q.items.size() * sizeof(ProcItem)));
        MFH_CUDA_CHECK(cudaMemcpyAsync(h->d_items, q.items.data(), q.items.size() * sizeof(ProcItem),
                                       cudaMemcpyHostToDevice, st));
    }
    {   // compact ascending slot lists per block row
        const int ns = std::max(q.n_slots, 1);
        std::vector<int32_t> lists((size_t)q.n_blk * (ns + 1), 0);
        for (int b = 0; b < q.n_blk; ++b) {
            int32_t* L = lists.data() + (size_t)b * (ns + 1);
            for (int sl = 0; sl < q.n_slots; ++sl)
                if (q.slot_valid[(size_t)b * q.n_slots + sl]) L[1 + L[0]++] = sl;
            if (b < q.row_first || b >= q.row_first + q.row_count) L[0] |= SLOT_SKIP_ROW;
            if (!q.own[(size_t)b * q.n_blk + b]) L[0] |= SLOT_NO_H0;
        }
        MFH_CUDA_CHECK(guarded_malloc(h, (void**)&h->d_slot_list, lists.size() * sizeof(int32_t)));
        MFH_CUDA_CHECK(cudaMemcpy(h->d_slot_list, lists.data(), lists.size() * sizeof(int32_t),
                                  cudaMemcpyHostToDevice));
    }
    if (!q.pair_items.empty()) {
        MFH_CUDA_CHECK(guarded_malloc(h, (void**)&h->d_pair_items, q.pair_items.size() * sizeof(ProcItem)));
        MFH_CUDA_CHECK(cudaMemcpyAsync(h->d_pair_items, q.pair_items.data(), q.pair_items.size() * sizeof(ProcItem),
                                       cudaMemcpyHostToDevice, st));
    }
    if (!q.tc_pairs.empty()) {   // two-sided tensor-core generator (k-vector complex64 plans)
        MFH_CUDA_CHECK(guarded_malloc(h, (void**)&h->d_tc_pairs, q.tc_pairs.size() * sizeof(int32_t)));
        MFH_CUDA_CHECK(cudaMemcpyAsync(h->d_tc_pairs, q.tc_pairs.data(), q.tc_pairs.size() * sizeof(int32_t), cudaMemcpyHostToDevice, st));
    }
    if (!q.tc_left.empty()) {
        MFH_CUDA_CHECK(guarded_malloc(h, (void**)&h->d_tc_left, q.tc_left.size() * sizeof(int32_t)));
        MFH_CUDA_CHECK(cudaMemcpyAsync(h->d_tc_left, q.tc_left.data(), q.tc_left.size() * sizeof(int32_t), cudaMemcpyHostToDevice, st));
    }
    if (!q.ct_left.empty()) {
        MFH_CUDA_CHECK(guarded_malloc(h, (void**)&h->d_ct_left, q.ct_left.size() * sizeof(int32_t)));
        MFH_CUDA_CHECK(cudaMemcpyAsync(h->d_ct_left, q.ct_left.data(), q.ct_left.size() * sizeof(int32_t), cudaMemcpyHostToDevice, st));
    }
    if (!q.tc_cpairs.empty()) {   // two-sided cached kernel (k-vector complex64 pair caches)
        MFH_CUDA_CHECK(guarded_malloc(h, (void**)&h->d_tc_cpairs, q.tc_cpairs.size() * sizeof(int32_t)));
        MFH_CUDA_CHECK(cudaMemcpyAsync(h->d_tc_cpairs, q.tc_cpairs.data(), q.tc_cpairs.size() * sizeof(int32_t), cudaMemcpyHostToDevice, st));
    }
    if (!q.tc_skip.empty()) {
        MFH_CUDA_CHECK(guarded_malloc(h, (void**)&h->d_tc_skip, q.tc_skip.size()));
        MFH_CUDA_CHECK(cudaMemcpyAsync(h->d_tc_skip, q.tc_skip.data(), q.tc_skip.size(), cudaMemcpyHostToDevice, st));
    }
    MFH_CUDA_CHECK(guarded_malloc(h, (void**)&h->d_counter, (3 + (size_t)q.n_blk) * sizeof(int32_t)));
    MFH_CUDA_CHECK(cudaMemsetAsync(h->d_counter, 0, (3 + (size_t)q.n_blk) * sizeof(int32_t), st));
    {   // fused tail (launch-bound regime): contributions the last-arrival reduce waits for per block row
        std::vector<int32_t> expected(q.n_blk, 0);
        for (const ProcItem& it : q.items) {
            ++expected[it.n];
            if (it.col_slot >= 0) ++expected[it.m];
        }
        MFH_CUDA_CHECK(guarded_malloc(h, (void**)&h->d_expected, expected.size() * sizeof(int32_t)));
        MFH_CUDA_CHECK(cudaMemcpy(h->d_expected, expected.data(), expected.size() * sizeof(int32_t), cudaMemcpyHostToDevice));
        h->fused_tail = q.mode == MFH_MODE_PROCEDURAL && q.k == 1 && q.part_world == 1 && !q.items.empty() &&
                        h->D <= kFusedTailMaxD;
    }
    MFH_CUDA_CHECK(guarded_malloc(h, (void**)&h->d_io, (size_t)2 * h->D * q.k * cb));
    MFH_CUDA_CHECK(cudaMemsetAsync(h->d_io, 0, (size_t)2 * h->D * q.k * cb, st));   // MFH_PART_ROWS leaves foreign rows untouched
    // scratch of the chained drivers, allocated here so that mfh_chebyshev* / mfh_lanczos_bounds never allocate
    // (they can be captured in a CUDA graph without a warm-up call)
    MFH_CUDA_CHECK(guarded_malloc(h, (void**)&h->d_cheb, cheb_scratch_bytes(h->D, h->dtype, q.k)));
    if (q.k == 1) MFH_CUDA_CHECK(guarded_malloc(h, (void**)&h->d_lanczos, lanczos_scratch_bytes(h->D, h->dtype)));
    if (h->kind == MFH_SRC_DIAG_PLUS_GUE) {
        MFH_CUDA_CHECK(guarded_malloc(h, (void**)&h->d_h0, (size_t)h->D * (h->dtype == MFH_C128 ? 8 : 4)));
        int rc = launch_h0(h, h->d_h0, st);
        if (rc) return rc;
    }
    int rc = ensure_gen_table(h, st);
    if (rc) return rc;
    if (h->kind == MFH_SRC_EXTERNAL) {   // the caller supplies the stored blocks (mfh_set_block)
        h->ext_set.assign((size_t)q.n_cached, 0);
        h->ext_missing = q.n_cached;
    } else {
        rc = launch_fill_cache(h, st);
        if (rc) return rc;
    }
    MFH_CUDA_CHECK(cudaStreamSynchronize(st));
    h->planned = true;
    return MFH_OK;
}

// ev: optional 4 events recorded before/between/after the three launches (mfh_apply_timed).
static int apply_impl(mfh_handle h, const void* psi, void* phi, const double* lambdas, cudaStream_t st,
                      cudaEvent_t* ev = nullptr)
{
    const Plan& p = h->plan;
    int rc, dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev != h->device) {
        set_error("the handle was planned on CUDA device %d, the current device is %d", h->device, dev);
        return MFH_ERR_BAD_STATE;
    }
    if (h->kind == MFH_SRC_EXTERNAL && h->ext_missing > 0) {
        set_error("external operator: %lld of %lld stored blocks have not been set (mfh_set_block)", (long long)h->ext_missing,
                  (long long)p.n_cached);
        return MFH_ERR_BAD_STATE;
    }
    if (ev) cudaEventRecord(ev[0], st);
    const bool overlap = partial_overlap_supported(h);   // cached and generated parts in one kernel (Eq. 33)
    if (!overlap && (rc = p.pairs ? launch_cached_pairs(h, psi, st) : launch_cached(h, psi, st))) return rc;
    if (ev) cudaEventRecord(ev[1], st);
    if (overlap) {
        if ((rc = launch_partial_overlap(h, psi, st))) return rc;
    } else if (p.k == 1) {
        const bool fused = h->fused_tail;   // the kernel reduces as well: one launch per apply
        if ((rc = launch_proc_single(h, psi, fused ? phi : nullptr, lambdas ? lambdas[0] : h->lambda, st))) return rc;
        if (fused) {
            if (ev) { cudaEventRecord(ev[2], st); cudaEventRecord(ev[3], st); }
            return MFH_OK;
        }
    } else if (p.slot_multi >= 0 && p.covered_blocks < p.owned_blocks) {
        if ((rc = launch_proc_multi(h, psi, st))) return rc;
    }
    if (ev) cudaEventRecord(ev[2], st);
    rc = launch_reduce(h, psi, phi, lambdas, st);
    if (ev) cudaEventRecord(ev[3], st);
    return rc;
}

// An apply inside a chain (Chebyshev, Lanczos): on a partitioned handle the result must be complete on
// every rank before the next O(D) update, so the registered exchange hook runs right after the apply.
static int apply_chained(mfh_handle h, const void* psi, void* phi, cudaStream_t st, const double* lambdas = nullptr)
{
    int rc = apply_impl(h, psi, phi, lambdas, st);
    if (rc || (h->part_world <= 1 && !h->exchange)) return rc;   // a registered hook also runs at world 1 (tests)
    if (!h->exchange) {
        set_error("partitioned handle (world %d): register an exchange hook with mfh_set_exchange", h->part_world);
        return MFH_ERR_BAD_STATE;
    }
    if (h->exchange(h->exchange_user, phi, (size_t)h->D * h->plan.k * complex_bytes(h->dtype), (void*)st)) {
        set_error("exchange hook failed");
        return MFH_ERR_CUDA;
    }
    return MFH_OK;
}

// Algorithm 2: time R_bench applies of a committed plan after R_warm warm-ups.
static int time_plan(mfh_handle h, cudaStream_t st, double& seconds)
{
    const int R_warm = 1, R_bench = 3;
    const size_t bytes = (size_t)h->D * h->plan.k * complex_bytes(h->dtype);
    char* psi = (char*)h->d_io;
    char* phi = psi + bytes;
    MFH_CUDA_CHECK(cudaMemsetAsync(psi, 0, bytes, st));   // timing does not depend on the values
    cudaEvent_t a, b;
    MFH_CUDA_CHECK(cudaEventCreate(&a));
    if (cudaEventCreate(&b) != cudaSuccess) {
        cudaEventDestroy(a);
        set_error("time_plan: cudaEventCreate failed");
        return MFH_ERR_CUDA;
    }
    int rc = MFH_OK;
    for (int r = 0; r < R_warm && !rc; ++r) rc = apply_impl(h, psi, phi, nullptr, st);
    cudaStreamSynchronize(st);
    cudaEventRecord(a, st);
    for (int r = 0; r < R_bench && !rc; ++r) rc = apply_impl(h, psi, phi, nullptr, st);
    cudaEventRecord(b, st);
    cudaError_t e = cudaStreamSynchronize(st);
    float ms = 0.f;
    cudaEventElapsedTime(&ms, a, b);
    cudaEventDestroy(a);
    cudaEventDestroy(b);
    if (rc) return rc;
    MFH_CUDA_CHECK(e);
    seconds = (double)ms * 1e-3 / R_bench;   // Eq. 21
    return MFH_OK;
}

}  // namespace mfh

using namespace mfh;

extern "C" {

MFH_API const char* mfh_last_error(void) { return g_err; }

MFH_API int mfh_create(mfh_handle* out, int64_t D, int32_t B, uint64_t seed, int32_t source_kind,
                       double lambda, int32_t dtype, uint64_t seed_h0)
{
    if (!out) { set_error("mfh_create: out is NULL"); return MFH_ERR_INVALID_ARG; }
    *out = nullptr;
    if (D < 32 || D > (int64_t)1 << 31 || D % 32 != 0) {
        set_error("mfh_create: D=%lld must be a multiple of 32 in [32, 2^31]", (long long)D);
        return MFH_ERR_INVALID_ARG;
    }
    if (B != 0 && !valid_B(D, B)) {
        set_error("mfh_create: B=%d must be a multiple of %d, <= %d, dividing D=%lld", B, MFH_MIN_B,
                  MFH_MAX_B, (long long)D);
        return MFH_ERR_INVALID_ARG;
    }
    if (source_kind < MFH_SRC_GUE || source_kind > MFH_SRC_EXTERNAL) {
        set_error("mfh_create: unknown source kind %d", source_kind);
        return MFH_ERR_INVALID_ARG;
    }
    if (dtype != MFH_C128 && dtype != MFH_C64) {
        set_error("mfh_create: unknown dtype %d", dtype);
        return MFH_ERR_INVALID_ARG;
    }
    if (!std::isfinite(lambda)) { set_error("mfh_create: lambda is not finite"); return MFH_ERR_INVALID_ARG; }
    mfh_handle h = new mfh_handle_s();
    h->D = D;
    h->B_req = B;
    h->seed = seed;
    h->seed_h0 = seed_h0;
    h->kind = source_kind;
    h->dtype = dtype;
    h->lambda = lambda;
    *out = h;
    return MFH_OK;
}

MFH_API int mfh_destroy(mfh_handle h)
{
    if (!h) return MFH_OK;
    free_plan_resources(h);
    for (cudaEvent_t e : h->timing_events) cudaEventDestroy(e);
    if (h->d_gen_tab) cudaFree(h->d_gen_tab);
    delete h;
    return MFH_OK;
}

MFH_API int mfh_set_source_params(mfh_handle h, const double* theta_host)
{
    if (!h || !theta_host) { set_error("mfh_set_source_params: NULL pointer"); return MFH_ERR_INVALID_ARG; }
    if (h->kind != MFH_SRC_ANALYTIC) { set_error("mfh_set_source_params: handle is not MFH_SRC_ANALYTIC"); return MFH_ERR_INVALID_ARG; }
    for (int q = 0; q < 6; ++q)
        if (!std::isfinite(theta_host[q])) { set_error("mfh_set_source_params: theta[%d] is not finite", q); return MFH_ERR_INVALID_ARG; }
    if (theta_host[1] < 0.0) { set_error("mfh_set_source_params: alpha must be >= 0"); return MFH_ERR_INVALID_ARG; }
    free_plan_resources(h);
    h->analytic.t = theta_host[0];
    h->analytic.alpha = theta_host[1];
    h->analytic.cphi = std::cos(theta_host[2]);
    h->analytic.sphi = std::sin(theta_host[2]);
    h->analytic.W = theta_host[3];
    h->analytic.beta2pi = 6.283185307179586476925 * theta_host[4];
    h->analytic.delta = theta_host[5];
    h->analytic_set = true;
    return MFH_OK;
}

MFH_API int mfh_set_block(mfh_handle h, int32_t n, int32_t m, const void* block, int32_t is_device, void* stream)
{
    if (!h || !block) { set_error("mfh_set_block: NULL pointer"); return MFH_ERR_INVALID_ARG; }
    if (h->kind != MFH_SRC_EXTERNAL) { set_error("mfh_set_block: handle is not MFH_SRC_EXTERNAL"); return MFH_ERR_INVALID_ARG; }
    if (!h->planned) { set_error("mfh_set_block: call mfh_plan first"); return MFH_ERR_BAD_STATE; }
    const Plan& p = h->plan;
    if (n < 0 || m < 0 || n >= p.n_blk || m >= p.n_blk) {
        set_error("mfh_set_block: block (%d,%d) outside %d x %d", n, m, p.n_blk, p.n_blk);
        return MFH_ERR_INVALID_ARG;
    }
    const int32_t slot = p.cache_slot[(size_t)n * p.n_blk + m];
    if (slot < 0) {
        set_error("mfh_set_block: block (%d,%d) is not stored by this plan (%s)", n, m,
                  slot == -2 ? "pair cache: pass the canonical block n <= m" : "owned by another rank");
        return MFH_ERR_INVALID_ARG;
    }
    cudaStream_t st = (cudaStream_t)stream;
    const size_t bytes = (size_t)p.B * p.B * complex_bytes(h->dtype);
    int rc;
    if (is_device) {
        rc = launch_store_block_at(h, slot, n, m, block, st);
    } else if (h->dtype == MFH_C64 && p.k > 1) {
        // tiled cache: stage on the device (one reusable block, freed with the plan), then re-lay
        if (!h->d_stage) MFH_CUDA_CHECK(guarded_malloc(h, (void**)&h->d_stage, bytes));
        MFH_CUDA_CHECK(cudaMemcpyAsync(h->d_stage, block, bytes, cudaMemcpyHostToDevice, st));
        rc = launch_store_block_at(h, slot, n, m, h->d_stage, st);
        MFH_CUDA_CHECK(cudaStreamSynchronize(st));   // the host block and the staging block may be reused
    } else {
        MFH_CUDA_CHECK(cudaMemcpyAsync((char*)h->d_cache + (size_t)slot * bytes, block, bytes, cudaMemcpyHostToDevice, st));
        MFH_CUDA_CHECK(cudaStreamSynchronize(st));   // the host block may be reused by the caller
        rc = MFH_OK;
    }
    if (rc) return rc;
    if (!h->ext_set[slot]) {
        h->ext_set[slot] = 1;
        --h->ext_missing;
    }
    return MFH_OK;
}

MFH_API int mfh_set_partition(mfh_handle h, int32_t rank, int32_t world, int32_t scheme)
{
    if (!h) { set_error("mfh_set_partition: NULL handle"); return MFH_ERR_INVALID_ARG; }
    if (world < 1 || rank < 0 || rank >= world || scheme < MFH_PART_NONE || scheme > MFH_PART_PAIRS ||
        (scheme == MFH_PART_NONE && world != 1)) {
        set_error("mfh_set_partition: invalid rank %d / world %d / scheme %d", rank, world, scheme);
        return MFH_ERR_INVALID_ARG;
    }
    free_plan_resources(h);   // a committed plan belongs to the previous partition
    h->part_rank = rank;
    h->part_world = world;
    h->part_scheme = world == 1 ? (int32_t)MFH_PART_NONE : scheme;
    return MFH_OK;
}

MFH_API int mfh_set_exchange(mfh_handle h, mfh_exchange_fn fn, void* user)
{
    if (!h) { set_error("mfh_set_exchange: NULL handle"); return MFH_ERR_INVALID_ARG; }
    h->exchange = fn;
    h->exchange_user = user;
    return MFH_OK;
}

MFH_API int mfh_get_partition_rows(mfh_handle h, int32_t* first_block_row, int32_t* n_block_rows, int32_t* B_out)
{
    if (!h || !first_block_row || !n_block_rows) { set_error("mfh_get_partition_rows: NULL pointer"); return MFH_ERR_INVALID_ARG; }
    if (!h->planned) { set_error("mfh_get_partition_rows: call mfh_plan first"); return MFH_ERR_BAD_STATE; }
    *first_block_row = h->plan.row_first;
    *n_block_rows = h->plan.row_count;
    if (B_out) *B_out = h->plan.B;
    return MFH_OK;
}

MFH_API int mfh_plan_analytic(int64_t D, int32_t dtype, int32_t k, int32_t mode, int32_t B,
                              int64_t n_applies_hint, int64_t hbm_free_bytes, char* json_out,
                              size_t json_cap)
{
    if (D < 32 || D % 32 != 0 || (dtype != MFH_C128 && dtype != MFH_C64) || k < 1 || k > MFH_MAX_K ||
        mode < MFH_MODE_AUTO || mode > MFH_MODE_PAIRS || (B != 0 && !valid_B(D, B)) || hbm_free_bytes <= 0) {
        set_error("mfh_plan_analytic: invalid argument");
        return MFH_ERR_INVALID_ARG;
    }
    std::vector<Candidate> cands;
    const double budget = planner_alpha() * (double)hbm_free_bytes;   // Eq. 18
    const int rc = enumerate_candidates(D, dtype, k, mode, B, n_applies_hint, budget, 148, cands);
    copy_json(plan_json(D, dtype, k, n_applies_hint, budget, 0, cands), json_out, json_cap);
    if (rc) set_error("mfh_plan_analytic: no candidate fits in %.0f bytes", budget);
    return rc;
}

MFH_API int mfh_plan_node_analytic(int64_t D, int32_t dtype, int32_t k, int32_t n_op, int64_t n_tasks, int32_t n_gpus,
                                   int64_t hbm_free_bytes_per_gpu, int32_t mode, int32_t B, int32_t scheme,
                                   int64_t n_applies_per_task, char* json_out, size_t json_cap)
{
    if (D < 32 || D % 32 != 0 || (dtype != MFH_C128 && dtype != MFH_C64) || k < 1 || k > MFH_MAX_K || n_op < 1 || n_op > 16 ||
        n_tasks < 1 || n_gpus < 1 || n_gpus > 1024 || hbm_free_bytes_per_gpu <= 0 || mode < MFH_MODE_AUTO || mode > MFH_MODE_PAIRS ||
        (B != 0 && !valid_B(D, B)) || (scheme != MFH_PART_ROWS && scheme != MFH_PART_PAIRS) || n_applies_per_task < 1) {
        set_error("mfh_plan_node_analytic: invalid argument");
        return MFH_ERR_INVALID_ARG;
    }
    std::string json;
    const int rc = plan_node(D, dtype, k, n_op, n_tasks, n_gpus, (double)hbm_free_bytes_per_gpu, mode, B, scheme,
                             n_applies_per_task, json);
    copy_json(json, json_out, json_cap);
    if (rc) set_error("mfh_plan_node_analytic: no row-group size has a plan that fits");
    return rc;
}

// Shared body of mfh_plan and mfh_plan_hybrid.  theta != nullptr: Algorithm 3, hybrid mode -- the memory-feasible
// candidates are ranked by the surrogate's t_NN(p) (Eq. 25), only the k_nn best are committed and timed (Algorithm 2),
// the best measured one is kept (Eq. 23).
static int plan_core(mfh_handle h, int32_t mode, int32_t k, int64_t n_applies_hint, int64_t hbm_budget_bytes, int32_t measure,
                     void* stream, char* json_out, size_t json_cap, const double* theta, int32_t hidden, int32_t k_nn)
{
    if (!h) { set_error("mfh_plan: NULL handle"); return MFH_ERR_INVALID_ARG; }
    if (k < 1 || k > MFH_MAX_K || mode < MFH_MODE_AUTO || mode > MFH_MODE_PAIRS || hbm_budget_bytes < 0) {
        set_error("mfh_plan: invalid argument (k=%d, mode=%d)", k, mode);
        return MFH_ERR_INVALID_ARG;
    }
    if (h->part_world > 1 && h->B_req == 0) {
        // block ownership is defined in block indices: ranks that picked different B would own sets that do not tile H
        set_error("mfh_plan: a partitioned handle (world %d) needs the block size fixed in mfh_create (B != 0): every "
                  "rank must plan the same B", h->part_world);
        return MFH_ERR_INVALID_ARG;
    }
    if (h->kind == MFH_SRC_EXTERNAL) {
        if (mode == MFH_MODE_AUTO) mode = MFH_MODE_FULL;
        if (mode != MFH_MODE_FULL && mode != MFH_MODE_PAIRS) {
            set_error("mfh_plan: external blocks need MFH_MODE_FULL or MFH_MODE_PAIRS (nothing can be generated)");
            return MFH_ERR_INVALID_ARG;
        }
        measure = 0;   // nothing to time before the blocks are there
    }
    if (h->kind == MFH_SRC_ANALYTIC && !h->analytic_set) {
        set_error("mfh_plan: MFH_SRC_ANALYTIC needs mfh_set_source_params first");
        return MFH_ERR_BAD_STATE;
    }
    cudaStream_t st = (cudaStream_t)stream;
    int dev = 0;
    MFH_CUDA_CHECK(cudaGetDevice(&dev));
    MFH_CUDA_CHECK(cudaDeviceGetAttribute(&h->sm_count, cudaDevAttrMultiProcessorCount, dev));
    free_plan_resources(h);   // a re-plan may reuse the memory of the previous plan
    if (dev != h->device) {   // the generator table and the kernel attributes belong to the previous device
        if (h->d_gen_tab) cudaFree(h->d_gen_tab);
        h->d_gen_tab = nullptr;
        h->gen_ready = false;
        h->smem_attr.clear();
        h->device = dev;
    }

    size_t free_b = 0, total_b = 0;
    MFH_CUDA_CHECK(cudaMemGetInfo(&free_b, &total_b));
    double budget = hbm_budget_bytes > 0 ? (double)hbm_budget_bytes : planner_alpha() * (double)free_b;
    budget = std::min(budget, 0.98 * (double)free_b);

    std::vector<Candidate> cands;
    Partition part;
    part.rank = h->part_rank;
    part.world = h->part_world;
    part.scheme = h->part_scheme;
    int rc = enumerate_candidates(h->D, h->dtype, k, mode, h->B_req, n_applies_hint, budget, h->sm_count, cands, part);
    if (rc) {
        copy_json(plan_json(h->D, h->dtype, k, n_applies_hint, budget, 0, cands), json_out, json_cap);
        set_error("mfh_plan: no candidate plan fits in %.0f bytes", budget);
        return rc;
    }
    auto make_plan = [&](const Candidate& c) {
        Plan p;
        p.B = c.B;
        p.k = k;
        p.cached_per_row = c.cached_per_row;
        p.pairs = c.pairs;
        p.stream_sms = c.stream_sms;
        p.part_rank = part.rank;
        p.part_world = part.world;
        p.part_scheme = part.scheme;
        p.allow_tc_pairs = c.tc_pairs;
        p.gen_two_sided = (h->kind != MFH_SRC_ANALYTIC);
        build_tables(p, h->D, h->dtype, h->sm_count);
        return p;
    };
    if (theta) {   // Algorithm 3: rank the feasible candidates by the surrogate's predicted apply time
        std::vector<double> x(MFH_SURROGATE_FEATURES);
        for (auto& c : cands) {
            if (!c.feasible) continue;
            rc = mfh_surrogate_features(h->D, h->dtype, k, c.mode, c.B, c.flops, c.cache_bytes, c.work_bytes, budget, 1, 1, 1,
                                        (double)total_b, h->sm_count, x.data());
            if (!rc) rc = mfh_surrogate_predict(theta, MFH_SURROGATE_FEATURES, hidden, x.data(), 1, &c.t_nn);
            if (rc) return rc;
        }
        std::stable_sort(cands.begin(), cands.end(), [](const Candidate& a, const Candidate& b) {
            if (a.feasible != b.feasible) return a.feasible;
            return a.feasible && a.t_nn < b.t_nn;
        });
    }
    if (measure) {   // Algorithm 2: K_bench best feasible candidates, argmin of the measured time
        const int K_bench = theta ? std::max(k_nn, 1) : 8;
        int tried = 0;
        for (auto& c : cands) {
            if (!c.feasible || tried >= K_bench) continue;
            ++tried;
            rc = commit_plan(h, make_plan(c), st);
            if (rc == MFH_ERR_OUT_OF_MEMORY) { c.feasible = false; continue; }
            if (rc) return rc;
            double s = 0.0;
            if ((rc = time_plan(h, st, s))) return rc;
            c.t_measured = s;
        }
        std::stable_sort(cands.begin(), cands.end(), [&](const Candidate& a, const Candidate& b) {
            const bool ma = a.t_measured >= 0, mb = b.t_measured >= 0;
            if (ma != mb) return ma;
            if (!ma) return false;
            const double n = (double)std::max<int64_t>(n_applies_hint, 1);
            return n * a.t_measured + a.t_fill < n * b.t_measured + b.t_fill;   // Eq. 22-23 with W = 1
        });
        if (cands.empty() || cands[0].t_measured < 0) {
            set_error("mfh_plan: no candidate could be committed");
            return MFH_ERR_OUT_OF_MEMORY;
        }
    }
    if (h->kind == MFH_SRC_EXTERNAL && cands[0].cached_fraction < 1.0) {
        if (mode == MFH_MODE_PAIRS && part.world > 1 && part.scheme == MFH_PART_ROWS) {
            set_error("mfh_plan: an external pair cache cannot be partitioned by rows (a pair split between two ranks is "
                      "stored by neither and nothing can be generated); use MFH_PART_PAIRS or MFH_MODE_FULL");
            return MFH_ERR_UNSUPPORTED;
        }
        set_error("mfh_plan: the external operator does not fit the budget as a %s cache", mode == MFH_MODE_PAIRS ? "pair" : "full");
        return MFH_ERR_OUT_OF_MEMORY;
    }
    rc = commit_plan(h, make_plan(cands[0]), st);
    if (rc) return rc;
    h->plan.json = plan_json(h->D, h->dtype, k, n_applies_hint, budget, theta ? 2 : measure, cands);
    copy_json(h->plan.json, json_out, json_cap);
    return MFH_OK;
}

MFH_API int mfh_plan(mfh_handle h, int32_t mode, int32_t k, int64_t n_applies_hint,
                     int64_t hbm_budget_bytes, int32_t measure, void* stream, char* json_out,
                     size_t json_cap)
{
    return plan_core(h, mode, k, n_applies_hint, hbm_budget_bytes, measure, stream, json_out, json_cap, nullptr, 0, 0);
}

MFH_API int mfh_plan_hybrid(mfh_handle h, const double* theta, int32_t hidden, int32_t k, int64_t n_applies_hint,
                            int64_t hbm_budget_bytes, int32_t k_nn, void* stream, char* json_out, size_t json_cap)
{
    if (!theta || hidden < 1 || k_nn < 1) { set_error("mfh_plan_hybrid: need theta, hidden >= 1, k_nn >= 1"); return MFH_ERR_INVALID_ARG; }
    return plan_core(h, MFH_MODE_AUTO, k, n_applies_hint, hbm_budget_bytes, 1, stream, json_out, json_cap, theta, hidden, k_nn);
}

MFH_API int mfh_get_plan(mfh_handle h, char* json_out, size_t json_cap)
{
    if (!h || !h->planned) { set_error("mfh_get_plan: handle not planned"); return MFH_ERR_BAD_STATE; }
    const Plan& p = h->plan;
    char buf[1024];
    snprintf(buf, sizeof buf,
             "{\"partition\":{\"scheme\":\"%s\",\"rank\":%d,\"world\":%d,\"owned_blocks\":%lld,\"first_block_row\":%d,\"block_rows\":%d},"
             "\"mode\":\"%s\",\"B\":%d,\"n_blk\":%d,\"k\":%d,\"cached_blocks\":%lld,\"cached_per_row\":%d,"
             "\"cached_fraction\":%.6g,\"cache_bytes\":%zu,\"work_bytes\":%zu,\"partial_slots\":%d,\"proc_items\":%zu,\"pair_items\":%zu,"
             "\"proc_rows_per_lane\":%d,\"proc_row_strips\":%d,\"stream_sms\":%d,\"two_sided_pairs\":%zu,\"two_sided_stored_pairs\":%zu,\"launches_per_apply\":%d}",
             p.part_scheme == MFH_PART_ROWS ? "rows" : (p.part_scheme == MFH_PART_PAIRS ? "pairs" : "none"), p.part_rank, p.part_world,
             (long long)p.owned_blocks, p.row_first, p.row_count,
             p.mode == MFH_MODE_FULL ? "full" : (p.mode == MFH_MODE_PARTIAL ? "partial" : (p.mode == MFH_MODE_PAIRS ? "pairs" : "procedural")), p.B,
             p.n_blk, p.k, (long long)p.n_cached, p.cached_per_row,
             (double)p.covered_blocks / (double)std::max<int64_t>(p.owned_blocks, 1), p.cache_bytes, p.work_bytes, p.n_slots,
             p.items.size(), p.pair_items.size(), p.R, p.Q, p.stream_sms, p.tc_pairs.size() / 2, p.tc_cpairs.size() / 3,
             h->fused_tail ? 1 : (partial_overlap_supported(h) ? 2 /* one kernel for both parts + reduce */
                                  : 1 + (p.n_cached > 0) + ((p.k == 1 && !p.items.empty()) ||
                                                            (p.k > 1 && p.covered_blocks < p.owned_blocks)) +
                                    // the two-sided k-vector generator and the one-sided kernel for what it leaves
                                    (p.k > 1 && !p.tc_pairs.empty() && tc_multi_supported(h) &&
                                     p.owned_blocks - p.covered_blocks - (int64_t)p.tc_pairs.size() > 0) +
                                    // stored pairs served by the two-sided cached kernel, next to the kernel for the diagonal blocks
                                    (p.k > 1 && !p.tc_cpairs.empty())));
    copy_json(buf, json_out, json_cap);
    return MFH_OK;
}

MFH_API int mfh_apply(mfh_handle h, const void* psi_dev, void* phi_dev, int32_t k,
                      const double* lambdas_host, void* stream)
{
    if (!h || !psi_dev || !phi_dev || psi_dev == phi_dev) {
        set_error("mfh_apply: NULL or aliased pointer");
        return MFH_ERR_INVALID_ARG;
    }
    if (!h->planned) { set_error("mfh_apply: call mfh_plan first"); return MFH_ERR_BAD_STATE; }
    if (k != h->plan.k) {
        set_error("mfh_apply: k=%d differs from the planned k=%d", k, h->plan.k);
        return MFH_ERR_INVALID_ARG;
    }
    cudaEvent_t* ev = nullptr;   // armed by mfh_timing_begin: events around the launches of this apply, no synchronisation
    if (h->timing_pos < h->timing_n) ev = h->timing_events.data() + 4 * (size_t)h->timing_pos++;
    return apply_impl(h, psi_dev, phi_dev, lambdas_host, (cudaStream_t)stream, ev);
}

static void timing_clear(mfh_handle h)
{
    for (cudaEvent_t e : h->timing_events) cudaEventDestroy(e);
    h->timing_events.clear();
    h->timing_n = h->timing_pos = 0;
}

MFH_API int mfh_timing_begin(mfh_handle h, int32_t n_applies)
{
    if (!h || n_applies < 1 || n_applies > 65536) { set_error("mfh_timing_begin: need a handle and 1 <= n_applies <= 65536"); return MFH_ERR_INVALID_ARG; }
    if (!h->planned) { set_error("mfh_timing_begin: call mfh_plan first"); return MFH_ERR_BAD_STATE; }
    timing_clear(h);
    h->timing_events.reserve(4 * (size_t)n_applies);
    for (int i = 0; i < 4 * n_applies; ++i) {
        cudaEvent_t e;
        if (cudaEventCreate(&e) != cudaSuccess) {
            timing_clear(h);
            set_error("mfh_timing_begin: cudaEventCreate failed");
            return MFH_ERR_CUDA;
        }
        h->timing_events.push_back(e);
    }
    h->timing_n = n_applies;
    return MFH_OK;
}

MFH_API int mfh_timing_end(mfh_handle h, float* ms_out, int32_t* n_recorded, void* stream)
{
    if (!h || !ms_out || !n_recorded) { set_error("mfh_timing_end: NULL pointer"); return MFH_ERR_INVALID_ARG; }
    const int n = h->timing_pos;
    cudaError_t e = cudaStreamSynchronize((cudaStream_t)stream);
    for (int a = 0; a < n && e == cudaSuccess; ++a) {
        cudaEvent_t* ev = h->timing_events.data() + 4 * (size_t)a;
        for (int i = 0; i < 3 && e == cudaSuccess; ++i) e = cudaEventElapsedTime(&ms_out[4 * a + i], ev[i], ev[i + 1]);
        if (e == cudaSuccess) e = cudaEventElapsedTime(&ms_out[4 * a + 3], ev[0], ev[3]);
    }
    *n_recorded = n;
    timing_clear(h);
    MFH_CUDA_CHECK(e);
    return MFH_OK;
}

MFH_API int mfh_apply_timed(mfh_handle h, const void* psi_dev, void* phi_dev, int32_t k,
                            const double* lambdas_host, void* stream, float* ms_out)
{
    if (!h || !psi_dev || !phi_dev || psi_dev == phi_dev || !ms_out) {
        set_error("mfh_apply_timed: NULL or aliased pointer");
        return MFH_ERR_INVALID_ARG;
    }
    if (!h->planned) { set_error("mfh_apply_timed: call mfh_plan first"); return MFH_ERR_BAD_STATE; }
    if (k != h->plan.k) { set_error("mfh_apply_timed: k mismatch"); return MFH_ERR_INVALID_ARG; }
    cudaStream_t st = (cudaStream_t)stream;
    cudaEvent_t ev[4];
    for (int i = 0; i < 4; ++i)
        if (cudaEventCreate(&ev[i]) != cudaSuccess) {
            while (i-- > 0) cudaEventDestroy(ev[i]);
            set_error("mfh_apply_timed: cudaEventCreate failed");
            return MFH_ERR_CUDA;
        }
    int rc = apply_impl(h, psi_dev, phi_dev, lambdas_host, st, ev);
    cudaError_t e = cudaStreamSynchronize(st);
    if (!rc && e == cudaSuccess) {
        for (int i = 0; i < 3; ++i) cudaEventElapsedTime(&ms_out[i], ev[i], ev[i + 1]);
        cudaEventElapsedTime(&ms_out[3], ev[0], ev[3]);
    }
    for (auto& x : ev) cudaEventDestroy(x);
    if (rc) return rc;
    MFH_CUDA_CHECK(e);
    return MFH_OK;
}

MFH_API int mfh_apply_host(mfh_handle h, const void* psi_host, void* phi_host, int32_t k,
                           const double* lambdas_host, void* stream)
{
    if (!h || !psi_host || !phi_host) { set_error("mfh_apply_host: NULL pointer"); return MFH_ERR_INVALID_ARG; }
    if (!h->planned) { set_error("mfh_apply_host: call mfh_plan first"); return MFH_ERR_BAD_STATE; }
    if (k != h->plan.k) { set_error("mfh_apply_host: k mismatch"); return MFH_ERR_INVALID_ARG; }
    cudaStream_t st = (cudaStream_t)stream;
    const size_t bytes = (size_t)h->D * k * complex_bytes(h->dtype);
    char* psi = (char*)h->d_io;
    char* phi = psi + bytes;
    MFH_CUDA_CHECK(cudaMemcpyAsync(psi, psi_host, bytes, cudaMemcpyHostToDevice, st));
    int rc = apply_impl(h, psi, phi, lambdas_host, st);
    if (rc) return rc;
    MFH_CUDA_CHECK(cudaMemcpyAsync(phi_host, phi, bytes, cudaMemcpyDeviceToHost, st));
    MFH_CUDA_CHECK(cudaStreamSynchronize(st));
    return MFH_OK;
}

// The Chebyshev series driver shared by the real- and imaginary-time entry points: terms l = 0..K-1 of
// out = phase * sum_l coef_l T_l(H~) psi with complex coefficients coef[l] = (re, im); K-1 chained applies.
static int chebyshev_series(mfh_handle h, const void* psi_dev, void* out_dev, double c, double R, int K,
                            const std::vector<double>& coef_re, const std::vector<double>& coef_im, double ph_re,
                            double ph_im, cudaStream_t st, const double* lambdas = nullptr)
{
    const size_t vb = (size_t)h->D * h->plan.k * complex_bytes(h->dtype);   // k columns: the O(D) updates are element-wise
    char* base = (char*)h->d_cheb;
    void *cur = base, *prev = base + vb, *acc = base + 2 * vb, *hq = base + 3 * vb;
    int rc;
    if ((rc = launch_cheb_first(h, psi_dev, cur, acc, coef_re[0], st))) return rc;      // Eq. 41 (coef_0 is real)
    for (int l = 1; l < K; ++l) {
        if ((rc = apply_chained(h, cur, hq, st, lambdas))) return rc;
        if ((rc = launch_cheb_step(h, hq, cur, prev, acc, c, 1.0 / R, l == 1, coef_re[l], coef_im[l], st))) return rc;   // Eq. 42-43
        std::swap(cur, prev);
    }
    return launch_cheb_final(h, acc, out_dev, ph_re, ph_im, st);
}

static int chebyshev_check(const char* fn, mfh_handle h, const void* psi_dev, const void* out_dev, double t, double e_min,
                           double e_max, double tol, bool any_k = false)
{
    if (!h || !psi_dev || !out_dev) { set_error("%s: NULL pointer", fn); return MFH_ERR_INVALID_ARG; }
    if (!h->planned) { set_error("%s: call mfh_plan first", fn); return MFH_ERR_BAD_STATE; }
    if (!any_k && h->plan.k != 1) { set_error("%s: plan with k = 1", fn); return MFH_ERR_INVALID_ARG; }
    if (!(e_max > e_min) || !std::isfinite(t) || !std::isfinite(e_min) || !std::isfinite(e_max) || !(tol > 0.0)) {
        set_error("%s: need e_max > e_min, finite t, tol > 0", fn);
        return MFH_ERR_INVALID_ARG;
    }
    return MFH_OK;
}

// J_l(x), l = 0..l_max, x >= 0, by downward recurrence J_{l-1} = (2l/x) J_l - J_{l+1} started far above both l_max
// and x (where J is negligible) and normalised with J_0 + 2 sum_{j>=1} J_{2j} = 1.  Stable for every x: the
// recurrence is followed in its growing direction.  (std::cyl_bessel_j switches to an asymptotic form that is wrong
// for x > 1000 at large order: J_500(1001) came out as -4e33.)
static void bessel_j_table(double x, int l_max, std::vector<double>& J)
{
    J.assign((size_t)l_max + 1, 0.0);
    if (x == 0.0) { J[0] = 1.0; return; }
    int start = std::max(l_max, (int)x) + 40 + (int)(12.0 * std::cbrt(std::max(x, 1.0)));
    start += start & 1;                                      // even
    double jp = 0.0, jc = 1e-300, norm = 0.0;                // J_{start+1}, J_start (arbitrary scale)
    std::vector<double> raw((size_t)l_max + 1, 0.0);
    for (int l = start; l >= 0; --l) {
        // jc = J_l (scaled)
        if (l <= l_max) raw[l] = jc;
        if (l == 0) norm += jc;
        else if ((l & 1) == 0) norm += 2.0 * jc;
        if (l > 0) {
            const double jm = (2.0 * l / x) * jc - jp;       // J_{l-1}
            jp = jc;
            jc = jm;
            if (std::fabs(jc) > 1e250) {                     // rescale before overflow
                jc *= 1e-250; jp *= 1e-250; norm *= 1e-250;
                for (double& r : raw) r *= 1e-250;
            }
        }
    }
    for (int l = 0; l <= l_max; ++l) J[l] = raw[l] / norm;
}

static int chebyshev_real_time(const char* fn, mfh_handle h, const void* psi_dev, void* out_dev, double t, double e_min,
                               double e_max, double tol, int32_t* n_terms_out, void* stream, const double* lambdas, bool any_k)
{
    int rc = chebyshev_check(fn, h, psi_dev, out_dev, t, e_min, e_max, tol, any_k);
    if (rc) return rc;
    const double c = 0.5 * (e_max + e_min), R = 0.5 * (e_max - e_min), a = R * t;
    // Bessel table J_l(|a|), l = 0..l_max (bessel_j_table below), K = 1 + last l with |J_l| >= tol.
    const double x = std::fabs(a);
    const int l_max = (int)(x + 80.0 + 12.0 * std::cbrt(x));
    std::vector<double> cr(l_max + 1, 0.0), ci(l_max + 1, 0.0), J;
    bessel_j_table(x, l_max, J);
    int K = 1;
    for (int l = 0; l <= l_max; ++l) {
        double v = J[l];
        if (!std::isfinite(v)) { set_error("%s: Bessel coefficient J_%d(%g) is not finite", fn, l, x); return MFH_ERR_NOT_CONVERGED; }
        if (a < 0 && (l & 1)) v = -v;
        if (std::fabs(v) >= tol) K = l + 1;
        if (l == 0) { cr[0] = v; continue; }
        switch (l & 3) {                                                            // 2 (-i)^l J_l
        case 0: cr[l] = 2.0 * v; break;
        case 1: ci[l] = -2.0 * v; break;
        case 2: cr[l] = -2.0 * v; break;
        case 3: ci[l] = 2.0 * v; break;
        }
    }
    if (K >= l_max) { set_error("%s: Bessel table too short", fn); return MFH_ERR_NOT_CONVERGED; }
    if (n_terms_out) *n_terms_out = K;
    return chebyshev_series(h, psi_dev, out_dev, c, R, K, cr, ci, std::cos(c * t), -std::sin(c * t), (cudaStream_t)stream, lambdas);
}

MFH_API int mfh_chebyshev(mfh_handle h, const void* psi_dev, void* out_dev, double t, double e_min,
                          double e_max, double tol, int32_t* n_terms_out, void* stream)
{
    return chebyshev_real_time("mfh_chebyshev", h, psi_dev, out_dev, t, e_min, e_max, tol, n_terms_out, stream, nullptr, false);
}

MFH_API int mfh_chebyshev_scan(mfh_handle h, const void* psi_dev, void* out_dev, double t, double e_min, double e_max,
                               double tol, const double* lambdas_host, int32_t* n_terms_out, void* stream)
{
    return chebyshev_real_time("mfh_chebyshev_scan", h, psi_dev, out_dev, t, e_min, e_max, tol, n_terms_out, stream, lambdas_host, true);
}

MFH_API int mfh_chebyshev_imag(mfh_handle h, const void* psi_dev, void* out_dev, double beta, double e_min,
                               double e_max, double tol, int32_t* n_terms_out, void* stream)
{
    int rc = chebyshev_check("mfh_chebyshev_imag", h, psi_dev, out_dev, beta, e_min, e_max, tol);
    if (rc) return rc;
    const double c = 0.5 * (e_max + e_min), R = 0.5 * (e_max - e_min), a = R * beta;
    if (beta < 0.0 || a > 600.0) {
        set_error("mfh_chebyshev_imag: need beta >= 0 and R beta <= 600 (got %g)", a);
        return MFH_ERR_INVALID_ARG;
    }
    // e^{-a} I_l(a) from the C++17 special function (the oracle uses Miller's recurrence); the scaled
    // values decrease monotonically in l.
    const int l_max = (int)(a + 60.0 + 12.0 * std::sqrt(a * 40.0 + 1.0));
    std::vector<double> cr(l_max + 1, 0.0), ci(l_max + 1, 0.0);
    const double ea = std::exp(-a);
    int K = 1;
    for (int l = 0; l <= l_max; ++l) {
        const double v = (a == 0.0) ? (l == 0 ? 1.0 : 0.0) : std::cyl_bessel_i((double)l, a) * ea;
        if (2.0 * v >= tol) K = l + 1;
        cr[l] = (l == 0 ? 1.0 : 2.0) * ((l & 1) ? -v : v);
    }
    if (K >= l_max) { set_error("mfh_chebyshev_imag: Bessel table too short"); return MFH_ERR_NOT_CONVERGED; }
    if (n_terms_out) *n_terms_out = K;
    return chebyshev_series(h, psi_dev, out_dev, c, R, K, cr, ci, 1.0, 0.0, (cudaStream_t)stream);
}

// Extreme eigenvalues of the symmetric tridiagonal T (diagonal a[0..m-1], off-diagonal b[0..m-2]) by
// Sturm-sequence bisection inside the Gershgorin interval (host; m <= a few hundred).
static void tridiag_extremes(const std::vector<double>& a, const std::vector<double>& b, int m, double& tmin, double& tmax)
{
    double lo = a[0], hi = a[0];
    for (int j = 0; j < m; ++j) {
        const double r = (j > 0 ? std::fabs(b[j - 1]) : 0.0) + (j < m - 1 ? std::fabs(b[j]) : 0.0);
        lo = std::min(lo, a[j] - r);
        hi = std::max(hi, a[j] + r);
    }
    auto count_below = [&](double x) {   // number of eigenvalues < x
        int cnt = 0;
        double q = a[0] - x;
        if (q < 0) ++cnt;
        for (int j = 1; j < m; ++j) {
            const double d = (q == 0.0) ? 1e-300 : q;
            q = a[j] - x - b[j - 1] * b[j - 1] / d;
            if (q < 0) ++cnt;
        }
        return cnt;
    };
    auto kth = [&](int kk) {   // kk-th smallest eigenvalue (0-based)
        double l = lo, h = hi;
        for (int it = 0; it < 200 && h - l > 4e-16 * std::max(std::fabs(l), std::fabs(h)); ++it) {
            const double mid = 0.5 * (l + h);
            if (count_below(mid) > kk) h = mid; else l = mid;
        }
        return 0.5 * (l + h);
    };
    tmin = kth(0);
    tmax = kth(m - 1);
}

MFH_API int mfh_lanczos_bounds(mfh_handle h, const void* psi_dev, int32_t m, double margin, double* e_min,
                               double* e_max, double* alpha_host, double* beta_host, void* stream)
{
    if (!h || !psi_dev || !e_min || !e_max) { set_error("mfh_lanczos_bounds: NULL pointer"); return MFH_ERR_INVALID_ARG; }
    if (m < 1 || m > 4096 || !(margin >= 0.0) || !std::isfinite(margin)) {
        set_error("mfh_lanczos_bounds: need 1 <= m <= 4096 and margin >= 0");
        return MFH_ERR_INVALID_ARG;
    }
    if (!h->planned) { set_error("mfh_lanczos_bounds: call mfh_plan first"); return MFH_ERR_BAD_STATE; }
    if (h->plan.k != 1) { set_error("mfh_lanczos_bounds: plan with k = 1"); return MFH_ERR_INVALID_ARG; }
    cudaStream_t st = (cudaStream_t)stream;
    m = (int32_t)std::min<int64_t>(m, h->D);
    const size_t vb = (size_t)h->D * complex_bytes(h->dtype);
    char* base = (char*)h->d_lanczos;
    void *v = base, *v_prev = base + vb, *w = base + 2 * vb;
    double* d_alpha = (double*)(base + 3 * vb);
    double* d_beta = d_alpha + 4096;
    double* d_norm0 = d_beta + 4096;
    double* d_partial = d_norm0 + 8;
    int rc;
    // v_1 = psi / ||psi||
    if ((rc = launch_lz_dot(h, psi_dev, psi_dev, d_partial, d_norm0, 1, st))) return rc;
    if ((rc = launch_lz_scale(h, psi_dev, v, d_norm0, st))) return rc;
    for (int j = 0; j < m; ++j) {
        if ((rc = apply_chained(h, v, w, st))) return rc;                                         // w = H v_j
        if ((rc = launch_lz_dot(h, v, w, d_partial, d_alpha + j, 0, st))) return rc;              // alpha_j = Re <v_j, w>
        if ((rc = launch_lz_update(h, w, v, v_prev, d_alpha + j, j ? d_beta + j - 1 : nullptr,    // w -= alpha v + beta v_prev
                                   d_partial, d_beta + j, st))) return rc;                        // beta_j = ||w||
        if ((rc = launch_lz_scale(h, w, v_prev, d_beta + j, st))) return rc;                      // v_{j+1} = w / beta_j
        std::swap(v, v_prev);
    }
    std::vector<double> a(m), b(m);
    MFH_CUDA_CHECK(cudaMemcpyAsync(a.data(), d_alpha, m * sizeof(double), cudaMemcpyDeviceToHost, st));
    MFH_CUDA_CHECK(cudaMemcpyAsync(b.data(), d_beta, m * sizeof(double), cudaMemcpyDeviceToHost, st));
    MFH_CUDA_CHECK(cudaStreamSynchronize(st));
    for (int j = 0; j < m; ++j)
        if (!std::isfinite(a[j]) || !std::isfinite(b[j])) {
            set_error("mfh_lanczos_bounds: breakdown at step %d (invariant subspace or zero start vector)", j);
            return MFH_ERR_NOT_CONVERGED;
        }
    double tmin, tmax;
    tridiag_extremes(a, b, m, tmin, tmax);
    const double c = 0.5 * (tmax + tmin), R = 0.5 * (tmax - tmin);
    *e_min = c - (1.0 + margin) * R;
    *e_max = c + (1.0 + margin) * R;
    if (alpha_host) memcpy(alpha_host, a.data(), m * sizeof(double));
    if (beta_host) memcpy(beta_host, b.data(), m * sizeof(double));
    return MFH_OK;
}

MFH_API int mfh_chebyshev_steps(mfh_handle h, const void* psi_dev, void* out_dev, double tau, int32_t n_steps,
                                double e_min, double e_max, double tol, int32_t* n_terms_out, void* stream)
{
    if (n_steps < 1) { set_error("mfh_chebyshev_steps: n_steps must be >= 1"); return MFH_ERR_INVALID_ARG; }
    if (!h || !psi_dev || !out_dev || psi_dev == out_dev) {
        set_error("mfh_chebyshev_steps: NULL or aliased pointer");
        return MFH_ERR_INVALID_ARG;
    }
    // out <- U(tau) psi, then out <- U(tau) out through the library's own ping-pong buffer
    int rc = mfh_chebyshev(h, psi_dev, out_dev, tau, e_min, e_max, tol, n_terms_out, stream);
    if (rc || n_steps == 1) return rc;
    const size_t vb = (size_t)h->D * complex_bytes(h->dtype);
    char* scratch = (char*)h->d_cheb + 4 * vb;   // fifth vector of the Chebyshev scratch (allocated below)
    for (int s = 1; s < n_steps; ++s) {
        MFH_CUDA_CHECK(cudaMemcpyAsync(scratch, out_dev, vb, cudaMemcpyDeviceToDevice, (cudaStream_t)stream));
        if ((rc = mfh_chebyshev(h, scratch, out_dev, tau, e_min, e_max, tol, nullptr, stream))) return rc;
    }
    return MFH_OK;
}

MFH_API int mfh_debug_philox(uint64_t seed, uint32_t stream_id, const uint32_t* i_dev,
                             const uint32_t* j_dev, int64_t n, uint32_t* words_dev, void* stream)
{
    if (n < 0 || (n > 0 && (!i_dev || !j_dev || !words_dev))) {
        set_error("mfh_debug_philox: invalid argument");
        return MFH_ERR_INVALID_ARG;
    }
    return launch_philox_debug(seed, stream_id, i_dev, j_dev, n, words_dev, (cudaStream_t)stream);
}

MFH_API int mfh_materialize_block(mfh_handle h, int32_t n, int32_t m, void* block_dev, void* stream)
{
    if (!h || !block_dev) { set_error("mfh_materialize_block: NULL pointer"); return MFH_ERR_INVALID_ARG; }
    if (h->kind == MFH_SRC_EXTERNAL) {
        set_error("mfh_materialize_block: an external operator has no generator (its blocks are the caller's, mfh_set_block)");
        return MFH_ERR_UNSUPPORTED;
    }
    const int32_t B = h->planned ? h->plan.B : h->B_req;
    if (B <= 0) { set_error("mfh_materialize_block: block size not fixed yet"); return MFH_ERR_BAD_STATE; }
    const int32_t n_blk = (int32_t)(h->D / B);
    if (n < 0 || m < 0 || n >= n_blk || m >= n_blk) {
        set_error("mfh_materialize_block: block (%d,%d) outside %d x %d", n, m, n_blk, n_blk);
        return MFH_ERR_INVALID_ARG;
    }
    return launch_fill_block(h, B, n, m, block_dev, (cudaStream_t)stream);
}

MFH_API int mfh_debug_poison(mfh_handle h, void* stream)
{
    if (!h || !h->planned) { set_error("mfh_debug_poison: handle not planned"); return MFH_ERR_BAD_STATE; }
    cudaStream_t st = (cudaStream_t)stream;
    const Plan& p = h->plan;
    MFH_CUDA_CHECK(cudaMemsetAsync(h->d_work, 0xFF, p.work_bytes, st));                                 // NaN in float and double
    MFH_CUDA_CHECK(cudaMemsetAsync(h->d_cheb, 0xFF, (size_t)5 * h->D * p.k * complex_bytes(h->dtype), st));
    return MFH_OK;
}

MFH_API int mfh_debug_corrupt_guard(mfh_handle h, int32_t buffer_index, int32_t after)
{
    if (!h || !h->planned) { set_error("mfh_debug_corrupt_guard: handle not planned"); return MFH_ERR_BAD_STATE; }
    if (buffer_index < 0 || buffer_index >= (int32_t)h->guarded.size()) {
        set_error("mfh_debug_corrupt_guard: buffer %d of %zu", buffer_index, h->guarded.size());
        return MFH_ERR_INVALID_ARG;
    }
    const auto& g = h->guarded[buffer_index];
    char* at = (char*)g.first + (after ? GUARD_BYTES + g.second : GUARD_BYTES - 1);   // first byte after / last byte before
    MFH_CUDA_CHECK(cudaMemset(at, 0, 1));
    return MFH_OK;
}

MFH_API int mfh_debug_selfcheck(mfh_handle h, int64_t* bad_guard_bytes, void* stream)
{
    if (!h || !bad_guard_bytes) { set_error("mfh_debug_selfcheck: NULL pointer"); return MFH_ERR_INVALID_ARG; }
    if (!h->planned) { set_error("mfh_debug_selfcheck: handle not planned"); return MFH_ERR_BAD_STATE; }
    cudaStream_t st = (cudaStream_t)stream;
    MFH_CUDA_CHECK(cudaStreamSynchronize(st));
    std::vector<unsigned char> buf(GUARD_BYTES);
    int64_t bad = 0;
    for (const auto& g : h->guarded)
        for (int side = 0; side < 2; ++side) {
            const char* src = (const char*)g.first + (side ? GUARD_BYTES + g.second : 0);
            MFH_CUDA_CHECK(cudaMemcpy(buf.data(), src, GUARD_BYTES, cudaMemcpyDeviceToHost));
            for (unsigned char c : buf) bad += (c != GUARD_BYTE);
        }
    *bad_guard_bytes = bad;
    return MFH_OK;
}

MFH_API int mfh_debug_bessel_j(double x, int32_t l_max, double* out_host)
{
    if (!out_host || l_max < 0 || l_max > (1 << 24) || !(x >= 0.0) || !std::isfinite(x)) {
        set_error("mfh_debug_bessel_j: need x >= 0 finite, 0 <= l_max <= 2^24, out != NULL");
        return MFH_ERR_INVALID_ARG;
    }
    std::vector<double> J;
    bessel_j_table(x, l_max, J);
    memcpy(out_host, J.data(), ((size_t)l_max + 1) * sizeof(double));
    return MFH_OK;
}

MFH_API int mfh_debug_h0(mfh_handle h, void* h0_dev, void* stream)
{
    if (!h || !h0_dev) { set_error("mfh_debug_h0: NULL pointer"); return MFH_ERR_INVALID_ARG; }
    return launch_h0(h, h0_dev, (cudaStream_t)stream);
}

}  // extern "C"

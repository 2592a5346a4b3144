// mfh_plan.cu -- single-GPU execution planner (host code).
//   Algorithm 1, analytic memory-constrained planning      P:258-296, Eq. 14-20
//   adaptive block size / cache budget                      P:409-446, Eq. 27
//   runtime model T = N_blk^2 [t_src + t_mv] (or the max)    P:533-547, Eq. 32-33; Eq. 36
// and the tables a committed plan needs: which blocks are cached, how the uncached block pairs
// are split into work items of the fused kernel, and which partial-sum slots feed each block row.
#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdlib>
#include "mfh_internal.cuh"
#include "mfh_plan.h"

namespace mfh {

// Model constants (seconds, bytes/s, generations/s).  Starting values; the measured planner
// (mfh_plan with measure != 0) overrides the ranking with device timings (Algorithm 2).
static const double kAlpha = 0.9;            // safety fraction of Eq. 18 (the paper gives none)
static const double kBwRead = 7.2e12;        // cached streaming, B/s (measured on C2: 7.3e12)
static const double kBwWrite = 3.0e12;       // cache fill stores, B/s
static const double kLaunch = 6e-6;          // per kernel launch

static double gen_pairs_per_s(int dtype) { return dtype == MFH_C128 ? 2.5e11 : 6.0e11; }   // measured on C4: 2.56e11
static double gen_entries_per_s(int dtype, int k)
{
    // one-sided generation plus 4k FMAs per entry on the same issue slots
    const double gen = dtype == MFH_C128 ? 1.6e11 : 5.0e11;
    const double mac = dtype == MFH_C128 ? 2.3e12 : 9.0e12;   // complex MACs/s (FP64 / FP32 FMA rate / 4)
    return 1.0 / (1.0 / gen + (double)k / mac);
}

// Read bandwidth of n SMs streaming alone (2 CTAs x 8 warps per SM, 16 x 128-bit loads in flight per lane), measured
// on one B200 with the other SMs idle: one SM pulls up to ~140 GB/s, 48 SMs already 6.0 TB/s, 64 SMs 7.0 TB/s
// (DESIGN.md 6.6).  Derated by 7 % for the strip loop's arithmetic and psi staging.
static double stream_bw_of_sms(int n, int sm_count)
{
    static const double pts[] = {0, 16, 32, 40, 48, 56, 64, 80, 96, 148};
    static const double gbs[] = {0, 2331, 4377, 5262, 6017, 6549, 6964, 7319, 7449, 7430};
    const double x = 148.0 * n / std::max(sm_count, 1);
    for (int i = 1; i < 10; ++i)
        if (x <= pts[i]) return 0.93e9 * (gbs[i - 1] + (gbs[i] - gbs[i - 1]) * (x - pts[i - 1]) / (pts[i] - pts[i - 1]));
    return 0.93e9 * gbs[9];
}

// Eq. 33 with the SMs partitioned between the two parts: n SMs stream the cached bytes, S - n generate;
// T(n) = max(bytes / BW(n), t_gen S / (S - n)).  Returns the n that minimises it and the time.
int choose_stream_sms(double cache_bytes, double t_gen_all_sms, int sm_count, double* t_out)
{
    int best = 1;
    double tb = 1e300;
    for (int n = 1; n < sm_count; ++n) {
        const double t = std::max(cache_bytes / stream_bw_of_sms(n, sm_count), t_gen_all_sms * sm_count / (double)(sm_count - n));
        if (t < tb) { tb = t; best = n; }
    }
    if (t_out) *t_out = tb;
    return best;
}

static void appendf(std::string& s, const char* fmt, ...)
{
    char buf[512];
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(buf, sizeof buf, fmt, ap);
    va_end(ap);
    s += buf;
}

static const char* mode_name(int mode)
{
    switch (mode) {
    case MFH_MODE_PROCEDURAL: return "procedural";
    case MFH_MODE_PARTIAL: return "partial";
    case MFH_MODE_FULL: return "full";
    case MFH_MODE_PAIRS: return "pairs";
    }
    return "auto";
}

// Offsets d = (m - n) mod N in the order 0, +1, -1, +2, -2, ...: a symmetric band around the
// diagonal, so that uncached blocks come in mirrored pairs the fused kernel generates once.
static std::vector<int> band_offsets(int N)
{
    std::vector<int> out;
    std::vector<char> seen(N, 0);
    for (int d = 0; (int)out.size() < N; ++d) {
        const int cand[2] = {((d % N) + N) % N, ((-d % N) + N) % N};
        for (int c : cand)
            if (!seen[c]) {
                seen[c] = 1;
                out.push_back(c);
            }
    }
    return out;
}

// Rows per lane R (row tile = 32 R rows) and row strips per block Q of the fused kernel.
// Prefer R = 4 (one psi_j load and one shuffle pair per 4 generated entries); go lower only when
// the block is too small or there would not be one item per resident CTA.  Q grows until there
// are ~24 items per SM (tail of the dynamic schedule below ~2 %) while the column-side partial
// slots (N_blk * Q vectors) stay small.
void choose_tiling(int B, int n_blk, int n_pairs, int sm_count, int& R, int& Q)
{
    R = 1;
    for (int r : {4, 2, 1}) {
        if (B % (32 * r) != 0) continue;
        R = r;
        // one item per resident CTA (2 per SM); a 5 % shortfall costs less than halving R (C1: R = 2 with 288
        // items on 296 slots runs in 57 us, R = 1 with 576 items in 68 us)
        if ((int64_t)n_pairs * (B / (32 * r)) >= 2LL * sm_count * 19 / 20) break;
    }
    const int qmax = B / (32 * R);
    Q = 1;
    while (qmax % (Q * 2) == 0 && (int64_t)n_pairs * Q < 48LL * sm_count && (int64_t)n_blk * Q * 2 <= 512) Q *= 2;
}

// Generator table of mfh_gen.cuh for dimension D (host arithmetic in long double).
void make_gen_table(int64_t D, GenHostD& out)
{
    const long double K2 = 1.0L / (long double)D;             // 2 s^2, s = 1/sqrt(2D)
    const long double LN2 = 0.693147180559945309417232121458L;
    const long double PI = 3.141592653589793238462643383280L;
    const int NL = 1 << GEN_LOG_BITS, NS = 1 << GEN_SC_BITS;
    for (int i = 0; i < NL; ++i) {
        const double inv = (double)(1.0L / (1.0L + ((long double)i + 0.5L) / NL));   // 1/c, then c := 1/inv exactly
        out.tab.tlog[i].x = inv;
        out.tab.tlog[i].y = (double)(K2 * logl((long double)inv));                   // -K2 ln c
    }
    for (int i = 0; i < NS; ++i) {
        const long double A = 2.0L * PI * (((long double)i + 0.5L) * 4194304.0L * (1024.0L / NS) + 0.5L) / 4294967296.0L;
        out.tab.tsc[i].x = (double)cosl(A);
        out.tab.tsc[i].y = (double)sinl(A);
    }
    for (int idx = 0; idx < 34; ++idx) out.tab.elog[idx] = (double)(K2 * (long double)(33 - idx) * LN2);
    out.gc.c1 = (double)(-K2);
    out.gc.c2 = (double)(K2 / 2.0L);
    out.gc.c3 = (double)(-K2 / 3.0L);
    out.gc.c4 = (double)(K2 / 4.0L);
    out.gc.ang = (double)(2.0L * PI / 4294967296.0L);
    out.gc.ang_off = -2097152.0 * out.gc.ang;   // exact: a power-of-two multiple of the rounded constant
}

// Offsets covered by a Hermitian pair cache with c band offsets: circular block distance < c.
int pair_full_offsets(int N) { return N / 2 + 1; }

// Ownership of the block positions under mfh_set_partition (R20).
void partition_mask(int N, const Partition& part, std::vector<uint8_t>& own)
{
    own.assign((size_t)N * N, part.world <= 1 ? 1 : 0);
    if (part.world <= 1) return;
    if (part.scheme == MFH_PART_ROWS) {
        // contiguous slabs of block rows (the paper's row sets R_j)
        const int lo = (int)((int64_t)N * part.rank / part.world), hi = (int)((int64_t)N * (part.rank + 1) / part.world);
        for (int n = lo; n < hi; ++n)
            for (int m = 0; m < N; ++m) own[(size_t)n * N + m] = 1;
        return;
    }
    // unordered pairs {n, n+d} dealt round-robin, nearest block diagonals first: each rank gets the same
    // mix of distances (so of cached and generated pairs) and a pair's two positions stay together
    int64_t idx = 0;
    for (int d = 0; d <= N / 2; ++d)
        for (int n = 0; n < N; ++n) {
            if (2 * d == N && n >= N / 2) continue;
            const int m = (n + d) % N;
            if (idx++ % part.world == part.rank) own[(size_t)n * N + m] = own[(size_t)m * N + n] = 1;
        }
}

void build_tables(Plan& p, int64_t D, int dtype, int sm_count)
{
    const int N = p.n_blk = (int)(D / p.B);
    const int c = p.cached_per_row;
    Partition part;
    part.rank = p.part_rank;
    part.world = p.part_world;
    part.scheme = p.part_scheme;
    partition_mask(N, part, p.own);
    auto own = [&](int n, int m) { return p.own[(size_t)n * N + m] != 0; };
    p.owned_blocks = 0;
    for (uint8_t o : p.own) p.owned_blocks += o;
    p.row_first = 0;
    p.row_count = N;
    if (part.world > 1 && part.scheme == MFH_PART_ROWS) {
        p.row_first = (int)((int64_t)N * part.rank / part.world);
        p.row_count = (int)((int64_t)N * (part.rank + 1) / part.world) - p.row_first;
    }
    p.cache_slot.assign((size_t)N * N, -1);
    for (int n = 0; n < N; ++n)
        for (int m = 0; m < N; ++m)
            if (!own(n, m)) p.cache_slot[(size_t)n * N + m] = -3;
    p.pair_items.clear();
    int n_stored = 0;
    if (!p.pairs) {
        // full blocks, row-balanced symmetric band (R5), owned positions only
        const std::vector<int> offs = band_offsets(N);
        for (int n = 0; n < N; ++n)
            for (int t = 0; t < c; ++t) {
                const int m = (n + offs[t]) % N;
                if (own(n, m)) p.cache_slot[(size_t)n * N + m] = n_stored++;
            }
    } else {
        // canonical pairs: every unordered block pair {n,m} with circular
        // distance d < c is stored once as block (min,max); the mirrored position is marked -2.
        // A pair split between two ranks (MFH_PART_ROWS) is not stored: both halves are generated.
        for (int d = 0; d < c && d <= N / 2; ++d)
            for (int n = 0; n < N; ++n) {
                const int m = (n + d) % N;
                if (d == 0) {
                    if (own(n, n)) p.cache_slot[(size_t)n * N + n] = n_stored++;
                    continue;
                }
                if (2 * d == N && n >= N / 2) continue;   // {n, n+N/2} was stored from the other side
                const int lo = std::min(n, m), hi = std::max(n, m);
                if (!own(lo, hi) || !own(hi, lo)) continue;
                p.cache_slot[(size_t)lo * N + hi] = n_stored++;
                p.cache_slot[(size_t)hi * N + lo] = -2;
            }
    }
    p.n_cached = n_stored;
    auto uncached = [&](int n, int m) { return p.cache_slot[(size_t)n * N + m] == -1; };
    int64_t covered = 0;
    for (int32_t v : p.cache_slot) covered += (v >= 0 || v == -2);
    p.covered_blocks = covered;

    p.pair_kind.assign((size_t)N * N, PAIR_NONE);
    p.items.clear();
    int n_pairs = 0;
    if (p.k == 1) {
        for (int n = 0; n < N; ++n) {
            if (uncached(n, n)) p.pair_kind[(size_t)n * N + n] = PAIR_DIAG;
            for (int m = n + 1; m < N; ++m) {
                const bool a = uncached(n, m), b = uncached(m, n);
                if (a && b) p.pair_kind[(size_t)n * N + m] = PAIR_TWO_SIDED;
                else if (a) p.pair_kind[(size_t)n * N + m] = PAIR_ONE_SIDED;
                else if (b) p.pair_kind[(size_t)m * N + n] = PAIR_ONE_SIDED;
            }
        }
        for (uint8_t kd : p.pair_kind) n_pairs += (kd != PAIR_NONE);
    }
    const int n_pair_blocks = p.pairs ? n_stored : 0;
    choose_tiling(p.B, N, std::max(n_pairs + n_pair_blocks, 1), sm_count, p.R, p.Q);

    // partial-sum slots: [cached rows] [row side, one per column block] [column side, one per
    // (row block, strip)] [k-vector kernel, one per column block]
    int s = 0;
    p.slot_cache = p.slot_row0 = p.slot_col0 = p.slot_multi = -1;
    if (!p.pairs && n_stored > 0 && p.k == 1) p.slot_cache = s++;
    if (p.k == 1 && n_pairs + n_pair_blocks > 0) {
        p.slot_row0 = s;
        s += N;
        p.slot_col0 = s;
        s += N * p.Q;
    }
    if (p.k > 1) {   // k-vector kernels (generated and cached blocks): one partial slot per column block m
        p.slot_multi = s;
        s += N;
    }
    // k-vector two-sided generator (complex64, mfh_tc.cu): a block pair whose two positions are both generated is
    // generated ONCE; its column side gets one slot per (row block, 128-row strip), like the one-vector kernel's
    p.tc_pairs.clear();
    p.tc_cpairs.clear();
    p.tc_skip.clear();
    p.slot_mcol0 = -1;
    p.pair_units = false;
    const int tcS = p.B / 128;
    if (p.allow_tc_pairs && tc_pairs_supported(dtype, p.k, p.B)) {
        // (partitioned handles: only pairs whose two positions this rank owns -- all of its pairs under MFH_PART_PAIRS,
        // the pairs inside its slab of block rows under MFH_PART_ROWS; uncached() is false for positions not owned)
        for (int n = 0; n < N; ++n)
            for (int m = n + 1; m < N; ++m) {
                if (p.gen_two_sided && uncached(n, m) && uncached(m, n)) {
                    p.tc_pairs.push_back(n);
                    p.tc_pairs.push_back(m);
                } else if (p.pairs && p.cache_slot[(size_t)n * N + m] >= 0 && p.cache_slot[(size_t)m * N + n] == -2) {
                    // stored pair: unit-image layout, both positions from one read (pairs_tc_kernel<true>)
                    p.tc_cpairs.push_back(n);
                    p.tc_cpairs.push_back(m);
                    p.tc_cpairs.push_back(p.cache_slot[(size_t)n * N + m]);
                }
            }
        p.pair_units = !p.tc_cpairs.empty();
        if (!p.tc_pairs.empty() || !p.tc_cpairs.empty()) {
            p.tc_skip.assign((size_t)N * N, 0);
            p.slot_mcol0 = s;
            s += N * tcS;
        }
    }
    p.n_slots = s;
    p.slot_valid.assign((size_t)N * std::max(s, 1), 0);
    auto valid = [&](int b, int slot) -> uint8_t& { return p.slot_valid[(size_t)b * p.n_slots + slot]; };
    for (int b = 0; b < N; ++b) {
        if (p.slot_cache >= 0) valid(b, p.slot_cache) = 1;
        if (p.slot_multi >= 0)
            for (int m = 0; m < N; ++m) valid(b, p.slot_multi + m) = own(b, m);   // nobody writes a block that is not ours
    }
    auto two_sided = [&](int n, int m) {
        p.tc_skip[(size_t)n * N + m] = p.tc_skip[(size_t)m * N + n] = 1;
        valid(m, p.slot_multi + n) = 0;   // position (m, n) arrives through the column-side slots instead
        for (int t = 0; t < tcS; ++t) valid(m, p.slot_mcol0 + n * tcS + t) = 1;
    };
    for (size_t q = 0; q + 1 < p.tc_pairs.size(); q += 2) two_sided(p.tc_pairs[q], p.tc_pairs[q + 1]);
    for (size_t q = 0; q + 2 < p.tc_cpairs.size(); q += 3) two_sided(p.tc_cpairs[q], p.tc_cpairs[q + 1]);
    p.ct_left.clear();
    if (!p.tc_cpairs.empty())
        for (int n = 0; n < N; ++n)
            for (int m = 0; m < N; ++m) {
                const int32_t cs = p.cache_slot[(size_t)n * N + m];
                if ((cs >= 0 || cs == -2) && !p.tc_skip[(size_t)n * N + m]) {
                    p.ct_left.push_back(n);
                    p.ct_left.push_back(m);
                }
            }
    p.tc_left.clear();
    if (!p.tc_pairs.empty())
        for (int n = 0; n < N; ++n)
            for (int m = 0; m < N; ++m)
                if (uncached(n, m) && !p.tc_skip[(size_t)n * N + m]) {
                    p.tc_left.push_back(n);
                    p.tc_left.push_back(m);
                }
    const int strip = p.B / p.Q;
    auto push_items = [&](std::vector<ProcItem>& dst, int n, int m, uint8_t kd) {
        valid(n, p.slot_row0 + m) = 1;
        const bool col = (kd == PAIR_TWO_SIDED || kd == PAIR_DIAG);
        for (int q = 0; q < p.Q; ++q) {
            ProcItem it;
            it.n = n;
            it.m = m;
            it.row0 = q * strip;
            it.nrows = strip;
            it.kind = kd;
            it.col_slot = (col && !(kd == PAIR_DIAG && &dst == &p.pair_items)) ? p.slot_col0 + n * p.Q + q : -1;
            if (it.col_slot >= 0) valid(m, it.col_slot) = 1;
            dst.push_back(it);
        }
    };
    if (p.k == 1 && n_pairs > 0) {
        // full-size two-sided items first, the half-size diagonal items last (better tail)
        for (int pass = 0; pass < 2; ++pass)
            for (int n = 0; n < N; ++n)
                for (int m = 0; m < N; ++m) {
                    const uint8_t kd = p.pair_kind[(size_t)n * N + m];
                    if (kd == PAIR_NONE || (pass == 0) != (kd != PAIR_DIAG)) continue;
                    push_items(p.items, n, m, kd);
                }
    }
    if (p.pairs && p.k == 1)   // stored blocks: off-diagonal pairs feed both sides, diagonal blocks the row side only
                               // (k-vector pair plans are served block by block by the tensor-core kernel)
        for (int n = 0; n < N; ++n)
            for (int m = n; m < N; ++m)
                if (p.cache_slot[(size_t)n * N + m] >= 0)
                    push_items(p.pair_items, n, m, n == m ? PAIR_DIAG : PAIR_TWO_SIDED);
    const size_t cb = complex_bytes(dtype);
    p.cache_bytes = (size_t)p.n_cached * p.B * p.B * cb;
    p.work_bytes = (size_t)std::max(p.n_slots, 1) * D * p.k * cb;
    if (covered == 0) p.mode = MFH_MODE_PROCEDURAL;
    else if (p.pairs) p.mode = MFH_MODE_PAIRS;
    else p.mode = (covered == p.owned_blocks ? MFH_MODE_FULL : MFH_MODE_PARTIAL);
}

// Scratch outside the partial slots: Chebyshev (5 k vectors), host-apply staging (2 k vectors), Lanczos (3 vectors
// + 80 KB of scalars, k = 1 plans), H0.
static size_t fixed_work_bytes(int64_t D, int dtype, int k)
{
    return (size_t)D * complex_bytes(dtype) * (7 * k + (k == 1 ? 3 : 0)) + (size_t)D * 8 + (k == 1 ? 81920 : 0);
}

Candidate evaluate_candidate(int64_t D, int dtype, int k, int B, int cached_per_row, bool pairs,
                             int64_t n_applies, int sm_count, const Partition& part, double budget_bytes)
{
    Candidate c;
    Plan p;
    p.B = B;
    p.k = k;
    p.cached_per_row = cached_per_row;
    p.pairs = pairs;
    p.part_rank = part.rank;
    p.part_world = part.world;
    p.part_scheme = part.scheme;
    c.pairs = pairs;
    build_tables(p, D, dtype, sm_count);
    if (budget_bytes >= 0 && (!p.tc_pairs.empty() || !p.tc_cpairs.empty()) &&
        (double)p.cache_bytes + (double)p.work_bytes + (double)fixed_work_bytes(D, dtype, k) > budget_bytes) {
        // the column-side slots of the two-sided k-vector generator do not fit: one-sided generation instead
        p.allow_tc_pairs = false;
        build_tables(p, D, dtype, sm_count);
    }
    c.tc_pairs = p.allow_tc_pairs;
    c.B = B;
    c.mode = p.mode;
    c.cached_per_row = cached_per_row;
    c.n_cached = p.n_cached;
    c.n_blk = p.n_blk;
    c.cache_bytes = (double)p.cache_bytes;                                   // M_op, Eq. 15-17
    c.work_bytes = (double)p.work_bytes + (double)fixed_work_bytes(D, dtype, k);   // M_work, Eq. 14
    const double cb = (double)complex_bytes(dtype);
    const double f = (double)p.covered_blocks / (double)std::max<int64_t>(p.owned_blocks, 1);   // entries served from the cache
    const double entries = (double)p.owned_blocks * B * B;                     // entries this rank applies
    c.cached_fraction = f;
    c.t_cached = c.cache_bytes / kBwRead;
    if (pairs && k > 1)
        // the mirrored positions cost a second pass: a second, transposed read of the stored blocks, or -- with the
        // unit-image layout -- the column side of the two-sided kernel, which reads every block once but is bound by
        // the tensor pipe and shared memory at the same time per stored byte (measured, C3: 1.25 ms for the pair cache
        // against 1.26 ms for the full cache)
        c.t_cached = (c.cache_bytes + (double)(p.covered_blocks - p.n_cached) * B * B * cb) / kBwRead;
    if (k == 1) {
        // generations: one per mirrored pair, one per one-sided entry, ~half of a diagonal block
        double gens = 0.0;
        for (uint8_t kd : p.pair_kind) {
            if (kd == PAIR_TWO_SIDED || kd == PAIR_ONE_SIDED) gens += (double)B * B;
            else if (kd == PAIR_DIAG) gens += 0.5 * (double)B * (B + 32.0 * p.R) + 0.5 * 32.0 * p.R * B;
        }
        double t = gens / gen_pairs_per_s(dtype);
        if (!p.items.empty()) {   // tail effect of whole-item scheduling
            const double slots = 2.0 * sm_count;
            const double waves = (double)p.items.size() / slots;
            t *= std::ceil(waves) / waves > 1.5 ? 1.5 : std::ceil(waves) / waves;
        }
        c.t_proc = t;
    } else {
        // the two-sided generator produces both positions of a pair from one generation
        const double gens = (1.0 - f) * entries - 0.5 * (double)p.tc_pairs.size() * B * B;
        c.t_proc = gens / gen_entries_per_s(dtype, k);
    }
    int launches = 1 + (p.n_cached > 0) + (p.covered_blocks < p.owned_blocks);
    c.t_reduce = (double)p.n_slots * 0.6 * D * k * cb / kBwRead;
    c.t_apply = c.t_cached + c.t_proc + c.t_reduce + launches * kLaunch;   // Eq. 32 (not overlapped)
    if (k == 1 && !pairs && p.n_cached > 0 && !p.items.empty()) {
        // one kernel, SMs partitioned between streaming and generating (Eq. 33: the max, not the sum)
        double t_max = 0.0;
        c.stream_sms = choose_stream_sms(c.cache_bytes, c.t_proc, sm_count, &t_max);
        c.t_apply = t_max + c.t_reduce + 2 * kLaunch;
    }
    const double stored = c.cache_bytes / cb;
    c.t_fill = stored / gen_entries_per_s(dtype, 0) + c.cache_bytes / kBwWrite;
    c.t_job = (double)std::max<int64_t>(n_applies, 1) * c.t_apply + c.t_fill;
    c.flops = 8.0 * entries * k;                                            // F_mv, Eq. 13 (this rank's share)
    return c;
}

static void candidate_json(std::string& s, const Candidate& c)
{
    appendf(s, "{\"mode\":\"%s\",\"B\":%d,\"n_blk\":%d,\"cached_blocks\":%lld,\"cached_per_row\":%d,",
            mode_name(c.mode), c.B, c.n_blk, (long long)c.n_cached, c.cached_per_row);
    appendf(s, "\"cached_fraction\":%.6g,", c.cached_fraction);
    appendf(s, "\"cache_bytes\":%.0f,\"work_bytes\":%.0f,\"total_bytes\":%.0f,\"feasible\":%s,",
            c.cache_bytes, c.work_bytes, c.cache_bytes + c.work_bytes, c.feasible ? "true" : "false");
    appendf(s, "\"model_apply_s\":%.6g,\"model_cached_s\":%.6g,\"model_proc_s\":%.6g,\"model_fill_s\":%.6g,"
               "\"model_job_s\":%.6g,\"flops_per_apply\":%.6g,\"measured_apply_s\":%.6g,\"surrogate_apply_s\":%.6g}",
            c.t_apply, c.t_cached, c.t_proc, c.t_fill, c.t_job, c.flops, c.t_measured, c.t_nn);
}

// Largest c in [0, c_max] with ok(c) (ok is monotone: more cached blocks need more memory); bisection,
// because every probe builds the plan tables.
template <typename F> static int largest_fitting(int c_max, F ok)
{
    if (c_max <= 0) return 0;
    if (ok(c_max)) return c_max;
    int lo = 0, hi = c_max;   // ok(lo) assumed (c = 0 caches nothing), !ok(hi)
    while (hi - lo > 1) {
        const int mid = lo + (hi - lo) / 2;
        if (ok(mid)) lo = mid; else hi = mid;
    }
    return lo;
}

int enumerate_candidates(int64_t D, int dtype, int k, int mode, int B_req, int64_t n_applies,
                         double budget_bytes, int sm_count, std::vector<Candidate>& out, const Partition& part)
{
    out.clear();
    std::vector<int> Bs;
    if (B_req > 0) Bs.push_back(B_req);
    else {
        // adaptive block size: powers of two dividing D, at most kMaxEnumBlocks block rows --
        // smaller blocks only add per-block overhead (Eq. 32), and the tables grow as N_blk^2
        const int kMaxEnumBlocks = 256;
        for (int B = MFH_MAX_B; B >= MFH_MIN_B; B /= 2)
            if (D % B == 0 && (D / B <= kMaxEnumBlocks || Bs.empty())) Bs.push_back(B);
    }
    const double cb = (double)complex_bytes(dtype);
    for (int B : Bs) {
        const int N = (int)(D / B);
        // cache budget -> cached blocks per row (Eq. 27 with full blocks; rows kept balanced)
        auto fits = [&](int c, bool pairs) {
            Candidate t = evaluate_candidate(D, dtype, k, B, c, pairs, n_applies, sm_count, part, budget_bytes);
            return t.cache_bytes + t.work_bytes <= budget_bytes;
        };
        std::vector<std::pair<int, bool>> cs;   // (cached_per_row or band offsets, pairs)
        if (mode == MFH_MODE_AUTO || mode == MFH_MODE_PROCEDURAL) cs.push_back({0, false});
        if (mode == MFH_MODE_AUTO || mode == MFH_MODE_FULL) cs.push_back({N, false});
        const bool pairs_ok = k == 1 ? B % (dtype == MFH_C128 ? 32 : 64) == 0 : tc_cached_multi_supported(dtype, k, B);
        if ((mode == MFH_MODE_AUTO || mode == MFH_MODE_PAIRS) && pairs_ok) {
            // Hermitian pair cache: the largest number of block diagonals that fits (Eq. 27 over
            // canonical pairs)
            int c = largest_fitting(pair_full_offsets(N), [&](int cc) { return fits(cc, true); });
            if (c > 0) cs.push_back({c, true});
            else if (mode == MFH_MODE_PAIRS) cs.push_back({1, true});   // reported as infeasible
        }
        if (mode == MFH_MODE_AUTO || mode == MFH_MODE_PARTIAL) {
            double room = budget_bytes - (double)fixed_work_bytes(D, dtype, k) - 3.0 * D * k * cb;
            int c = (int)std::floor(room * std::max(part.world, 1) / ((double)B * B * cb * N));   // a rank stores ~c N / world blocks
            c = largest_fitting(std::min(c, N - 1), [&](int cc) { return fits(cc, false); });
            if (c > 0) cs.push_back({c, false});
            // The overlapped kernel (complex128, one vector) shares every SM between the cached and the generated
            // part, and "as much as fits" is not its optimum (C5: 146 GB cached 31.4 ms, 100 GB 29.1 ms): two
            // smaller caches are offered as well; the analytic model (Eq. 32, a sum) ranks them below the largest,
            // the measured pass (Algorithm 2) decides.
            if (dtype == MFH_C128 && k == 1)
                for (int cc : {(3 * c) / 4, (3 * c) / 5})
                    if (cc > 0 && cc < c) cs.push_back({cc, false});
        }
        for (auto [c, pairs] : cs) {
            Candidate cand = evaluate_candidate(D, dtype, k, B, c, pairs, n_applies, sm_count, part, budget_bytes);
            cand.feasible = (cand.cache_bytes + cand.work_bytes <= budget_bytes);   // Eq. 18
            // cached k-vector blocks: B % 128 == 0 (tensor-core kernel for complex64, FP64 CUDA-core kernel for complex128)
            if (k > 1 && c > 0 && !(pairs ? tc_cached_multi_supported(dtype, k, B)
                                          : (tc_cached_multi_supported(dtype, k, B) || cached_multi_c128_supported(dtype, k, B))))
                cand.feasible = false;
            out.push_back(cand);
        }
    }
    std::stable_sort(out.begin(), out.end(), [](const Candidate& a, const Candidate& b) {
        if (a.feasible != b.feasible) return a.feasible;
        return a.t_job < b.t_job;
    });
    return (!out.empty() && out[0].feasible) ? MFH_OK : MFH_ERR_OUT_OF_MEMORY;
}

std::string plan_json(int64_t D, int dtype, int k, int64_t n_applies, double budget, int measured,
                      const std::vector<Candidate>& cands)
{
    std::string s;
    appendf(s, "{\"D\":%lld,\"dtype\":\"%s\",\"k\":%d,\"n_applies_hint\":%lld,\"budget_bytes\":%.0f,"
               "\"alpha\":%.2f,\"planner\":\"%s\",\"dense_bytes\":%.0f,\"chosen\":",
            (long long)D, dtype == MFH_C128 ? "c128" : "c64", k, (long long)n_applies, budget, kAlpha,
            measured == 2 ? "hybrid" : (measured ? "measured" : "analytic"), (double)D * D * complex_bytes(dtype));
    if (!cands.empty()) candidate_json(s, cands[0]);
    else s += "null";
    s += ",\"candidates\":[";
    for (size_t i = 0; i < cands.size(); ++i) {
        if (i) s += ",";
        candidate_json(s, cands[i]);
    }
    s += "]}";
    return s;
}

double planner_alpha() { return kAlpha; }

// Exchange step of a row group (all-gather or all-reduce of D k B_c bytes over NVLink 5 / NVSwitch): a
// latency term plus the bytes a rank receives at a conservative 400 GB/s.
static double exchange_seconds(int64_t D, int dtype, int k, int p_row)
{
    if (p_row <= 1) return 0.0;
    const double bytes = (double)D * k * complex_bytes(dtype);
    return 20e-6 + bytes * (double)(p_row - 1) / p_row / 400e9;
}

int plan_node(int64_t D, int dtype, int k, int n_op, int64_t n_tasks, int n_gpus, double free_per_gpu, int mode, int B_req,
              int scheme, int64_t n_applies_per_task, std::string& json)
{
    const double budget = kAlpha * free_per_gpu / n_op;   // Eq. 18, the operators share the memory evenly
    struct Row {
        int p_row, groups;
        int64_t waves;
        bool feasible;
        Candidate c;
        double t_apply, score;
    };
    std::vector<Row> rows;
    int best = -1;
    for (int p_row = 1; p_row <= n_gpus; ++p_row) {
        if (n_gpus % p_row) continue;
        Row r;
        r.p_row = p_row;
        r.groups = n_gpus / p_row;                                        // C(p)
        r.waves = (n_tasks + r.groups - 1) / r.groups;                     // Eq. 19
        Partition part;
        part.rank = 0;
        part.world = p_row;
        part.scheme = p_row > 1 ? scheme : (int)MFH_PART_NONE;
        std::vector<Candidate> cands;
        const int rc = enumerate_candidates(D, dtype, k, mode, B_req, r.waves * n_applies_per_task, budget, 148, cands, part);
        r.feasible = (rc == MFH_OK);
        if (!cands.empty()) r.c = cands[0];
        r.t_apply = r.feasible ? n_op * (r.c.t_apply + exchange_seconds(D, dtype, k, p_row)) : 0.0;
        r.score = r.feasible ? (double)r.waves * ((double)n_applies_per_task * r.t_apply + n_op * r.c.t_fill / std::max<int64_t>(r.waves, 1)) : 0.0;
        if (r.feasible && (best < 0 || r.score < rows[best].score)) best = (int)rows.size();
        rows.push_back(r);
    }
    auto row_json = [&](const Row& r) {
        appendf(json, "{\"p_row\":%d,\"groups\":%d,\"waves\":%lld,\"strategy\":\"%s\",\"feasible\":%s,", r.p_row, r.groups,
                (long long)r.waves, r.p_row == 1 ? "parameter-parallel" : (r.p_row == n_gpus ? "row-parallel" : "hybrid"),
                r.feasible ? "true" : "false");
        appendf(json, "\"mode\":\"%s\",\"B\":%d,\"operator_bytes_per_gpu\":%.0f,\"work_bytes_per_gpu\":%.0f,"
                      "\"total_bytes_per_gpu\":%.0f,\"model_apply_s\":%.6g,\"score_s\":%.6g}",
                mode_name(r.c.mode), r.c.B, n_op * r.c.cache_bytes, n_op * r.c.work_bytes,
                n_op * (r.c.cache_bytes + r.c.work_bytes), r.t_apply, r.score);
    };
    appendf(json, "{\"D\":%lld,\"dtype\":\"%s\",\"k\":%d,\"n_op\":%d,\"n_tasks\":%lld,\"n_gpus\":%d,\"alpha\":%.2f,"
                  "\"budget_bytes_per_gpu\":%.0f,\"scheme\":\"%s\",\"flops_per_apply\":%.6g,\"chosen\":",
            (long long)D, dtype == MFH_C128 ? "c128" : "c64", k, n_op, (long long)n_tasks, n_gpus, kAlpha, kAlpha * free_per_gpu,
            scheme == MFH_PART_ROWS ? "rows" : "pairs", 8.0 * n_op * (double)D * (double)D * k);
    if (best >= 0) row_json(rows[best]);
    else json += "null";
    json += ",\"row_groups\":[";
    for (size_t i = 0; i < rows.size(); ++i) {
        if (i) json += ",";
        row_json(rows[i]);
    }
    json += "]}";
    return best >= 0 ? MFH_OK : MFH_ERR_OUT_OF_MEMORY;
}

}  // namespace mfh

// mfh_tc.cu -- k-vector fused generate-and-apply on the 5th-generation tensor cores (complex64).
//
// Coupling scans (Eq. 12; BASELINE.json configs[2]): Phi = V Psi for k <= 16 vectors is a
// genuine dense contraction [128 x 16 columns of V] x [16 x 32] per tile, where the 32 real output
// columns are (Re Phi_v, Im Phi_v).  Each V entry is generated ONCE in registers (Philox + SFU
// Box-Muller, mfh_gen.cuh), split into two TF32 words (hi + lo) and written with tcgen05.st straight
// into TENSOR MEMORY as the A operand (lane = row, column = k index): the matrix never touches
// shared memory or HBM.  The B operands (psi, split the same way) are 2 KB shared-memory images
// in the canonical no-swizzle K-major UMMA layout.  One lane issues tcgen05.mma.kind::tf32 (A from
// TMEM, B from shared memory) with the [128 x 32] fp32 accumulator also in TMEM, so the 64 FFMA
// per entry of the CUDA-core kernel disappear from the issue slots that bound it.
// 3xTF32: D += A_hi B_hi + A_hi B_lo + A_lo B_hi (single-pass TF32 gives 2.9e-4 relative L2 and
// fails the 1e-4 tolerance; measured here: 9.5e-6 on C3, dominated by the tensor core's fp32
// accumulation over 1024 columns).  Complex arithmetic as two real operand pairs:
//     [Re Phi | Im Phi] += Re V x [Re Psi | Im Psi]  +  Im V x [-Im Psi | Re Psi].
// Warp-specialised CTA: 8 generator warps + 1 MMA warp, a 3-stage ring of (A columns in TMEM,
// B images in shared memory) guarded by mbarriers: generators wait on empty[s] (tcgen05.commit of
// the MMAs that read the stage), fill it, fence and arrive on full[s]; the MMA warp waits on
// full[s], issues 8 MMAs (see TC_ACC_COLS) and commits.  A CTA owns 128 rows x one column block m; the epilogue
// reads the accumulator with tcgen05.ld and writes the partial slot of column block m (added in
// index order by the reduce kernel).
#include <algorithm>
#include "mfh_internal.cuh"

namespace mfh {

constexpr int TC_GEN_WARPS = 8;               // generator warps; warp 8 builds the B operands and issues the MMAs
constexpr int TC_THREADS = 32 * (TC_GEN_WARPS + 1);
constexpr int TC_TP = 128;                    // rows per CTA = MMA M
constexpr int TC_TQ = 16;                     // columns per tile = TQ/8 MMA K-steps
constexpr int TC_NG = TC_TQ / 8;              // 4-column groups per generator thread and tile
constexpr int TC_N = 32;                      // MMA N: 16 vectors x (re, im)
constexpr int TC_B_TILE = TC_N * TC_TQ * 4;   // bytes of one B operand image in shared memory (2 KB)
constexpr int TC_STAGE = 4 * TC_B_TILE;       // B1_hi B1_lo B2_hi B2_lo
constexpr int TC_STAGES = 3;
// TMEM columns: [0,64) accumulator (two halves, see TC_ACC_COLS); stage s holds the four A images Er_hi Er_lo Ei_hi Ei_lo, 16 columns each
constexpr int TC_TMEM_COLS = (2 * TC_N + TC_STAGES * 4 * TC_TQ) <= 128 ? 128 : 256;
constexpr int TC_A_COL0 = 2 * TC_N;
constexpr int TC_A_STAGE_COLS = 4 * TC_TQ;
constexpr int TC_SBO = (TC_TQ / 4) * 128;     // byte stride between 8-row groups (A) / 8-column groups (B)
constexpr int TC_LBO = 128;                   // byte stride between the two 16-byte K halves of one MMA

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

// Shared-memory matrix descriptor, K-major, SWIZZLE_NONE: core matrix = 8 rows x 16 bytes.
__device__ __forceinline__ uint64_t umma_desc(uint32_t addr)
{
    return (uint64_t)((addr >> 4) & 0x3fffu) | ((uint64_t)(TC_LBO >> 4) << 16) | ((uint64_t)(TC_SBO >> 4) << 32) |
           (1ull << 46);
}

__device__ __forceinline__ uint64_t umma_desc_sbo(uint32_t addr, int sbo)
{
    return (uint64_t)((addr >> 4) & 0x3fffu) | ((uint64_t)(TC_LBO >> 4) << 16) | ((uint64_t)(sbo >> 4) << 32) |
           (1ull << 46);
}

// Instruction descriptor: D = F32, A = B = TF32, both K-major, M = 128, N = 32 or 64.
constexpr uint32_t tc_idesc(int n)
{
    return (1u << 4) | (2u << 7) | (2u << 10) | ((uint32_t)(n >> 3) << 17) | ((uint32_t)(TC_TP >> 4) << 24);
}
// 3xTF32 with two instructions per operand pair: the hi and lo images of B are adjacent in shared memory
// (8 row groups of one stride), so  A_hi x [B_hi | B_lo]  is ONE N = 64 MMA into accumulator columns
// [0,32) and [32,64), and  A_lo x B_hi  one N = 32 MMA into [0,32); the epilogue adds the two halves.
// The small MMAs of this kernel cost a fixed ~100 clocks each, so their number is what matters.
constexpr int TC_ACC_COLS = 2 * TC_N;

// A operand from TMEM (128 lanes x 8 columns), B from shared memory.
template <int N>
__device__ __forceinline__ void umma_tf32_ts(uint32_t d_tmem, uint32_t a_tmem, uint64_t b, uint32_t accumulate)
{
    asm volatile(
        "{\n\t"
        ".reg .pred p;\n\t"
        "setp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::tf32 [%0], [%1], %2, %3, p;\n\t"
        "}\n" ::"r"(d_tmem),
        "r"(a_tmem), "l"(b), "r"(tc_idesc(N)), "r"(accumulate)
        : "memory");
}

// Four consecutive TMEM columns of this thread's lane (warp-collective: lanes 32 (warp % 4) ..).
__device__ __forceinline__ void tmem_st4(uint32_t taddr, float a, float b, float c, float d)
{
    asm volatile("tcgen05.st.sync.aligned.32x32b.x4.b32 [%0], {%1, %2, %3, %4};" ::"r"(taddr), "r"(__float_as_uint(a)),
                 "r"(__float_as_uint(b)), "r"(__float_as_uint(c)), "r"(__float_as_uint(d))
                 : "memory");
}

// One elected lane of a converged warp (elect.sync): unlike `lane == 0` the compiler knows that exactly one thread is
// active, so the warp-uniform tcgen05 instructions inside need no per-instruction election loop.
__device__ __forceinline__ bool elect_one()
{
    uint32_t pred;
    asm volatile(
        "{\n\t"
        ".reg .pred p;\n\t"
        "elect.sync _|p, 0xffffffff;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t"
        "}\n"
        : "=r"(pred));
    return pred != 0;
}

__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity)
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
            : "r"(smem_u32(bar)), "r"(parity)
            : "memory");
    } while (!done);
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void umma_commit(uint64_t* bar)
{
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(bar))
                 : "memory");
}

// x = hi + lo with hi = x rounded to the nearest TF32 (integer add + mask: cvt.rna.tf32 costs four
// instructions with its NaN handling, and no entry is NaN or Inf); lo = x - hi is exact and the tensor
// core drops its low 13 bits (2^-22 of x).  Plain truncation of hi would bias every product one way.
__device__ __forceinline__ void split_tf32(float x, float& hi, float& lo)
{
    hi = __uint_as_float((__float_as_uint(x) + 0x1000u) & 0xffffe000u);
    lo = x - hi;
}

// Epilogue of warp w < 4: TMEM lanes 32w..32w+31 hold rows 32w + lane of the [128 x 32] accumulator
// (columns 0..15 real parts, 16..31 imaginary parts of the k vectors); dst = this row's k outputs.
__device__ __forceinline__ void tc_epilogue_load(uint32_t d_tmem, int w, float (&acc)[32])
{
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
#pragma unroll
    for (int half = 0; half < 2; ++half) {   // columns [0,32): A_hi B_hi + A_lo B_hi;  [32,64): A_hi B_lo
        uint32_t r[32];
        const uint32_t taddr = d_tmem + ((uint32_t)(32 * w) << 16) + 32 * half;
        asm volatile(
            "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
            "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
            "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
            : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]),
              "=r"(r[8]), "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]),
              "=r"(r[16]), "=r"(r[17]), "=r"(r[18]), "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]),
              "=r"(r[24]), "=r"(r[25]), "=r"(r[26]), "=r"(r[27]), "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31])
            : "r"(taddr)
            : "memory");
        asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
        for (int c = 0; c < 32; ++c) acc[c] = half ? acc[c] + __uint_as_float(r[c]) : __uint_as_float(r[c]);
    }
}
__device__ __forceinline__ void tc_epilogue_store(const float (&acc)[32], float2* dst, int k)
{
#pragma unroll
    for (int vv = 0; vv < 16; ++vv)
        if (vv < k) dst[vv] = make_float2(acc[vv], acc[16 + vv]);
}
__device__ __forceinline__ void tc_epilogue(uint32_t d_tmem, int w, float2* dst, int k)
{
    float acc[32];
    tc_epilogue_load(d_tmem, w, acc);
    tc_epilogue_store(acc, dst, k);
}

struct TcParams {
    GenArgs<float> G;
    int32_t B, n_blk, k, slot_multi;
    int64_t D;
    const int32_t* cache_slot;
    const uint8_t* skip;   // [n_blk*n_blk] positions served by the two-sided generator (nullptr: none)
    const int32_t* pos;    // compact list of the (row block, column block) positions to run (blockIdx.y), or nullptr: all
    const float2* psi;   // [D][k]
    float2* work;        // [n_slots][D][k]
};

// The 8 entries of one generator thread in one tile: row i, column groups gsel and gsel + 2.
template <int REL>
__device__ __forceinline__ void tc_tile_entries(const GenArgs<float>& G, uint32_t i, uint32_t j0, int gsel, float (&rh)[2][4],
                                                float (&rl)[2][4], float (&ih)[2][4], float (&il)[2][4])
{
#pragma unroll
    for (int gg = 0; gg < 2; ++gg)
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            const uint32_t j = j0 + 4 * (gsel + 2 * gg) + e;
            float hr, hi;
            if (REL > 0) entry_upper<float>(G, nullptr, i, j, hr, hi);
            else if (REL < 0) entry_lower<float>(G, nullptr, i, j, hr, hi);
            else entry_any<float>(G, nullptr, i, j, hr, hi);
            // A_hi = the value itself (the tensor core reads its TF32 part), A_lo = x - trunc(x), exact
            rh[gg][e] = hr;
            rl[gg][e] = hr - __uint_as_float(__float_as_uint(hr) & 0xffffe000u);
            ih[gg][e] = hi;
            il[gg][e] = hi - __uint_as_float(__float_as_uint(hi) & 0xffffe000u);
        }
}

// Generator warps (8 x 32 threads).  Per tile of 128 rows x 16 columns a thread produces the two
// 4-column groups g, g + 2 of row p (8 entries, one 16-byte store per operand image and group) and
// one (column, vector) element of the four psi images, then one lane per warp arrives on full[s].
// REL > 0: every entry has i < j (block above the diagonal), REL < 0: i > j, REL == 0: diagonal block.
template <int REL>
__device__ __forceinline__ void tc_generate(const TcParams& P, unsigned char* smem, uint64_t* full,
                                            uint64_t* empty, uint32_t d_tmem, uint32_t i_base, int m)
{
    const int tid = threadIdx.x, lane = tid & 31;
    const int p = tid & (TC_TP - 1), gsel = tid >> 7;
    const uint32_t i = i_base + p;
    const uint32_t a_lane = d_tmem + ((uint32_t)(p & ~31) << 16);   // this warp's 32 TMEM lanes: rows 32 (warp % 4) ..
    // (vector, column) of this thread's psi element: a warp covers 8 vectors x 4 columns = 32 distinct banks of a B image
    const int v = (tid & 7) | ((tid >> 2) & 8), qb = ((tid >> 3) & 3) | ((tid >> 6) << 2), k = P.k;
    // psi element (n, q) of a K-major B image: n = v (real part rows) and n = 16 + v (imaginary part rows)
    const int o_re = ((v & 7) * 16 + (v >> 3) * TC_SBO + (qb >> 2) * 128 + (qb & 3) * 4) / 4;
    const int o_im = o_re + 2 * TC_SBO / 4;
    const int n_tiles = P.B / TC_TQ;
    for (int t = 0; t < n_tiles; ++t) {
        const int s = t % TC_STAGES, u = t / TC_STAGES;
        const uint32_t j0 = (uint32_t)m * P.B + t * TC_TQ;
        const float2 x = (v < k && qb < TC_TQ) ? P.psi[(size_t)(j0 + qb) * k + v] : float2{0.f, 0.f};   // consumed after the entries
        float rh[TC_NG][4], rl[TC_NG][4], ih[TC_NG][4], il[TC_NG][4];
        if (REL != 0) tc_tile_entries<REL>(P.G, i, j0, gsel, rh, rl, ih, il);
        // diagonal block: only the tiles that cross the diagonal need the general rule (8 of B/16 per 128-row strip)
        else if (j0 >= i_base + TC_TP) tc_tile_entries<1>(P.G, i, j0, gsel, rh, rl, ih, il);
        else if (j0 + TC_TQ <= i_base) tc_tile_entries<-1>(P.G, i, j0, gsel, rh, rl, ih, il);
        else tc_tile_entries<0>(P.G, i, j0, gsel, rh, rl, ih, il);
        float prh, prl, pih, pil;
        split_tf32(x.x, prh, prl);
        split_tf32(x.y, pih, pil);
        if (u > 0) mbar_wait(&empty[s], (u - 1) & 1);   // the MMAs that read stage s have completed
        unsigned char* st = smem + s * TC_STAGE;
#pragma unroll
        for (int gg = 0; gg < TC_NG; ++gg) {   // A images: 4 columns of this thread's TMEM lane (= row p) per image
            const uint32_t ta = a_lane + (uint32_t)(TC_A_COL0 + s * TC_A_STAGE_COLS + 4 * (gsel + 2 * gg));
            tmem_st4(ta + 0 * TC_TQ, rh[gg][0], rh[gg][1], rh[gg][2], rh[gg][3]);
            tmem_st4(ta + 1 * TC_TQ, rl[gg][0], rl[gg][1], rl[gg][2], rl[gg][3]);
            tmem_st4(ta + 2 * TC_TQ, ih[gg][0], ih[gg][1], ih[gg][2], ih[gg][3]);
            tmem_st4(ta + 3 * TC_TQ, il[gg][0], il[gg][1], il[gg][2], il[gg][3]);
        }
        if (qb < TC_TQ) {   // B1 = [Re Psi | Im Psi], B2 = [-Im Psi | Re Psi]
            float* b = reinterpret_cast<float*>(st);
            constexpr int BT = TC_B_TILE / 4;
            b[0 * BT + o_re] = prh;  b[0 * BT + o_im] = pih;     // B1_hi
            b[1 * BT + o_re] = prl;  b[1 * BT + o_im] = pil;     // B1_lo
            b[2 * BT + o_re] = -pih; b[2 * BT + o_im] = prh;     // B2_hi
            b[3 * BT + o_re] = -pil; b[3 * BT + o_im] = prl;     // B2_lo
        }
        asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // generic-proxy writes -> async proxy (UMMA)
        asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
        __syncwarp();
        if (lane == 0) mbar_arrive(&full[s]);
    }
}

// MMA warp: waits for the 8 generator warps, issues the 8 MMAs of the tile from one lane and commits
// them onto empty[s] (the arrival that lets the generators overwrite the stage).
__device__ __forceinline__ void tc_mma_warp(const TcParams& P, unsigned char* smem, uint64_t* full, uint64_t* empty,
                                            uint64_t* done, uint32_t d_tmem)
{
    const int lane = threadIdx.x & 31;
    const int n_tiles = P.B / TC_TQ;
    for (int t = 0; t < n_tiles; ++t) {
        const int s = t % TC_STAGES, u = t / TC_STAGES;
        mbar_wait(&full[s], u & 1);
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        if (elect_one()) {
            const uint32_t b0 = smem_u32(smem + s * TC_STAGE);
            const uint32_t a0 = d_tmem + (uint32_t)(TC_A_COL0 + s * TC_A_STAGE_COLS);
#pragma unroll
            for (int ks = 0; ks < TC_TQ / 8; ++ks) {
                const uint32_t ko = ks * 2 * TC_LBO;
                const uint32_t er_h = a0 + 0 * TC_TQ + 8 * ks, er_l = a0 + 1 * TC_TQ + 8 * ks;
                const uint32_t ei_h = a0 + 2 * TC_TQ + 8 * ks, ei_l = a0 + 3 * TC_TQ + 8 * ks;
                const uint64_t b1 = umma_desc(b0 + 0 * TC_B_TILE + ko);   // [B1_hi | B1_lo] for N = 64, B1_hi for N = 32
                const uint64_t b2 = umma_desc(b0 + 2 * TC_B_TILE + ko);
                umma_tf32_ts<64>(d_tmem, er_h, b1, (t | ks) != 0);
                umma_tf32_ts<32>(d_tmem, er_l, b1, 1);
                umma_tf32_ts<64>(d_tmem, ei_h, b2, 1);
                umma_tf32_ts<32>(d_tmem, ei_l, b2, 1);
            }
            umma_commit(&empty[s]);                            // arrives when every MMA issued so far has completed
            if (t == n_tiles - 1) umma_commit(done);
        }
        __syncwarp();
    }
}

__global__ void __launch_bounds__(TC_THREADS, 2) proc_multi_tc_kernel(const TcParams P)
{
    extern __shared__ __align__(128) unsigned char smem[];
    __shared__ __align__(8) uint64_t full[TC_STAGES], empty[TC_STAGES], done;
    __shared__ uint32_t s_tmem;
    const int tid = threadIdx.x, w = tid >> 5;
    const int m = P.pos ? P.pos[2 * blockIdx.y + 1] : (int)blockIdx.y;
    const uint32_t i_base = (P.pos ? (uint32_t)P.pos[2 * blockIdx.y] * P.B : 0u) + blockIdx.x * TC_TP;
    const int n = (int)(i_base / (uint32_t)P.B);
    if (P.cache_slot[n * P.n_blk + m] != -1) return;   // cached block: not this kernel's
    if (P.skip && P.skip[n * P.n_blk + m]) return;     // served for both sides by pairs_tc_kernel

    if (tid == 0) {
        for (int s = 0; s < TC_STAGES; ++s) {
            mbar_init(&full[s], TC_GEN_WARPS);
            mbar_init(&empty[s], 1);
        }
        mbar_init(&done, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (w == TC_GEN_WARPS) {   // the MMA warp allocates 32 TMEM columns for the [128 x 32] fp32 accumulator
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&s_tmem)),
                     "n"(TC_TMEM_COLS)
                     : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const uint32_t d_tmem = s_tmem;

    if (w == TC_GEN_WARPS) tc_mma_warp(P, smem, full, empty, &done, d_tmem);
    else if (n < m) tc_generate<1>(P, smem, full, empty, d_tmem, i_base, m);
    else if (n > m) tc_generate<-1>(P, smem, full, empty, d_tmem, i_base, m);
    else tc_generate<0>(P, smem, full, empty, d_tmem, i_base, m);

    if (w < 4) {
        mbar_wait(&done, 0);
        tc_epilogue(d_tmem, w, P.work + ((size_t)(P.slot_multi + m) * P.D + i_base + 32 * w + (tid & 31)) * P.k, P.k);
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if (w == TC_GEN_WARPS)
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(d_tmem), "n"(TC_TMEM_COLS) : "memory");
}

// --------------------------------------------------------------------------------------------
// Two-sided k-vector generator (complex64): "generates ... each V block once" AND uses the Hermitian structure
// (Eq. 11): for a block pair n < m whose two positions are both generated, every entry
// V_ij (i in block n, j in block m) is generated ONCE and used for  Phi_i += V_ij Psi_j  (row side: the tile is the
// TMEM A operand as in the one-sided kernel, here in the cached kernel's interleaved (re, im) layout, see
// t2_psi_image) and for  Phi_j += conj(V_ij) Psi_i  (column side).  pairs_tc_kernel<true> is the same kernel for
// STORED pairs of a pair cache: the generator warps become converters of unit images landed by bulk copies.
//
// The column side contracts over the tile's ROWS, which are the lanes of the row side's A operand, so it cannot
// reuse that operand.  It swaps the operand roles instead: the generated tile is the B operand in shared memory,
//     B[n = column c][k' = (row r, part)] = (Re V_rc, Im V_rc),      K-major, 128-byte swizzle,
// written by the generator threads straight from their registers (raw value = TF32 hi part as the tensor core reads
// it, and a second image x - trunc(x)), and the strip's psi rows are the A operand, resident in TMEM for the whole
// item (a strip of 128 rows x all columns of the block):
//     A[(op, v)][k' = (r, part)]:  op = Re:  (Re Psi_rv,  Im Psi_rv);   op = Im:  (Im Psi_rv, -Re Psi_rv).
// 128 rows x 2 parts = 256 k' would need 256 TMEM columns; the strip's two 64-row halves are stacked in the LANES
// instead (lanes 0-63: rows 0-63, lanes 64-127: rows 64-127; inside a half: 32 lanes hi image, 32 lanes lo image)
// and the B operand lists the tile's columns twice (N = 64: columns for the first half of the rows, then for the
// second half), so one MMA does two K-steps' worth of useful work in the two diagonal quadrants of its [128 x 64]
// result and the other two quadrants are never read.  A unit = two tiles (32 columns): 16 K-steps x (raw, lo)
// = 32 MMAs of N = 64; its [128 x 64] accumulator is read out by four epilogue warps, the four quadrant pieces
// (hi/lo x row halves) are added through shared memory and written to the column-side partial slot of
// (row block, strip) -- a fixed order, no atomics.
//
// One persistent CTA per SM (all 512 TMEM columns): 16 generator warps in two groups that take the tiles
// alternately (thread = half a row of a tile, as in the one-sided kernel), 4 epilogue warps (they also build the
// psi operand of the NEXT item into the other of two TMEM buffers), 2 sum warps, one warp issuing the row-side MMAs,
// one the column-side MMAs (+ a bulk-copy producer warp in the cached variant).
// --------------------------------------------------------------------------------------------
constexpr int T2_GEN_WARPS = 16;
constexpr int T2_W_EPI = T2_GEN_WARPS;            // warps 16..19: TMEM lane quadrants 0..3
// Warp w runs on scheduler w % 4.  The MMA issuers sit on schedulers 2 and 3; two more warps on schedulers 0 and 1, fed
// through shared memory, do the cross-quadrant sums and the stores of the column side.  That keeps the epilogue warps'
// loop short (the column-side MMA warp waits for them before every unit: measured 17 % of its time when they also
// summed and stored) and spreads the helper instructions over the four schedulers (a generator warp on a busier
// scheduler makes the other 15 wait at every unit).
constexpr int T2_W_SUM = T2_GEN_WARPS + 4;        // warps 20, 21: cross-quadrant sums and stores of the column side
constexpr int T2_W_DMMA = T2_GEN_WARPS + 6;       // row-side MMA issuer (allocates TMEM)
constexpr int T2_W_MMMA = T2_GEN_WARPS + 7;       // column-side MMA issuer
constexpr int T2_THREADS = 32 * (T2_GEN_WARPS + 8);
constexpr int T2_COL_DACC = 0;                    // row-side accumulator [128 x 64] (TC_ACC_COLS)
constexpr int T2_COL_MACC = 64;                   // column-side accumulator [128 x 64]
constexpr int T2_COL_PSI = 128;                   // psi operand of the column side, two buffers (item parity) of 128 columns = (row % 64, part)
constexpr int T2_COL_ASTAGE = 384;                // row-side A stage of each group: 64 columns
constexpr int T2_UNIT_COLS = 32;                  // columns per unit (two tiles)
constexpr int T2_IMG = 128 * T2_UNIT_COLS * 8;    // one image (raw or lo) of a unit: 32 KB
constexpr int T2_UNIT = 2 * T2_IMG;
constexpr int T2_XCH = 4 * 32 * 32 * 4;           // epilogue exchange: [quadrant][column][lane] floats
constexpr int T2_SMEM = 1024 + 2 * T2_UNIT + 2 * TC_STAGE + 2 * T2_XCH;
// cached variant (stored pair blocks instead of generated ones): a producer warp, TMA stages of raw unit images
constexpr int T2C_W_TMA = T2_GEN_WARPS + 8;
constexpr int T2C_THREADS = 32 * (T2_GEN_WARPS + 9);
constexpr int T2C_STAGES = 3;
constexpr int T2C_SMEM = 1024 + T2C_STAGES * T2_IMG + 2 * T2_IMG + 2 * TC_STAGE + 2 * T2_XCH;

struct T2Params {
    GenArgs<float> G;
    int32_t B, n_blk, k, slot_multi, slot_mcol0, S, n_items, pstride;
    int64_t D;
    const int32_t* pairs;   // (row block, column block[, cache slot]) per pair, pstride ints each
    const float2* cache;    // cached variant: stored blocks in the unit-image layout (mfh_internal.cuh unit_image_offset)
    const float2* psi;
    float2* work;
};

struct T2Bars {
    uint64_t dfull[2], dempty[2];         // row-side stage of group g
    uint64_t mfull[2], mempty[2];         // unit buffers
    uint64_t macc_full, macc_empty;       // column-side accumulator
    uint64_t psi_full;                    // psi operand of the item in TMEM
    uint64_t ddone, dacc_empty;           // row-side accumulator
    uint64_t raw_full[T2C_STAGES], raw_empty[T2C_STAGES];   // cached variant: TMA stages of raw unit images
};

// K-major, SWIZZLE_128B: rows of 128 bytes (32 TF32), 8-row groups 1 KB apart.
__device__ __forceinline__ uint64_t umma_desc_sw128(uint32_t addr)
{
    return (uint64_t)((addr >> 4) & 0x3fffu) | (1ull << 16) | ((uint64_t)(1024 >> 4) << 32) | (1ull << 46) | (2ull << 61);
}

__device__ __forceinline__ void tmem_ld32(uint32_t taddr, uint32_t (&r)[32])
{
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
        "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
        "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
        : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]),
          "=r"(r[8]), "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]),
          "=r"(r[16]), "=r"(r[17]), "=r"(r[18]), "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]),
          "=r"(r[24]), "=r"(r[25]), "=r"(r[26]), "=r"(r[27]), "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31])
        : "r"(taddr)
        : "memory");
    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
}

// Row side of the two-sided kernels: INTERLEAVED operand layout (the cached kernel's, 6.5): K index k' = 2 c + part, so
// a thread's (re, im) pairs go to TMEM and to the column side's shared-memory image from the same register pairs.
// A stage: [A_hi: 32 columns][A_lo: 32 columns]; psi images B_hi | B_lo adjacent (N = 64 for A_hi, N = 32 for A_lo):
//   row v:      (Re Psi_cv, -Im Psi_cv) at k' = (2c, 2c+1)   -> Re Phi;   row 16 + v: (Im Psi_cv, Re Psi_cv) -> Im Phi.
constexpr int T2_BT = TC_N * 32 * 4;          // one psi image: 32 rows x 32 k' floats = 4 KB (T2_BT x 2 = TC_STAGE)
constexpr int T2_BSBO = (32 / 4) * 128;       // 1 KB between 8-row groups of a psi image
__device__ __forceinline__ void t2_psi_image(unsigned char* stage, int v, int qb, float2 x)
{
    float* b = reinterpret_cast<float*>(stage);
    const int o_re = ((v & 7) * 16 + (v >> 3) * T2_BSBO + (qb >> 1) * 128 + (qb & 1) * 8) / 4;
    const int o_im = o_re + 2 * T2_BSBO / 4;
    float prh, prl, pih, pil;
    split_tf32(x.x, prh, prl);
    split_tf32(x.y, pih, pil);
    *reinterpret_cast<float2*>(b + o_re) = make_float2(prh, -pih);
    *reinterpret_cast<float2*>(b + o_im) = make_float2(pih, prh);
    *reinterpret_cast<float2*>(b + T2_BT / 4 + o_re) = make_float2(prl, -pil);
    *reinterpret_cast<float2*>(b + T2_BT / 4 + o_im) = make_float2(pil, prl);
}

// Generator group g (256 threads): tiles 2u + g of every unit u.  Row side exactly as tc_generate<+1>; column side:
// the thread's 8 entries of row p go to the unit buffer as (Re, Im) pairs at
//   [(p % 64) / 16] 8 KB  +  [p / 64] 4 KB  +  [column / 8] 1 KB  +  [column % 8] 128 B  +  16-byte chunk ((p % 16) / 2) ^ (column % 8)  +  (p % 2) 8 B
// -- 16 lanes cover one 128-byte row, so the stores are conflict-free.
__device__ __forceinline__ void t2_generate(const T2Params& P, unsigned char* ubuf, unsigned char* bimg, T2Bars& bar, uint32_t d_tmem)
{
    const int tid = threadIdx.x, lane = tid & 31;
    const int g = tid >> 8, lt = tid & 255;
    const int p = lt & (TC_TP - 1), gsel = lt >> 7;
    const uint32_t a_lane = d_tmem + ((uint32_t)(p & ~31) << 16);
    // (vector, column) of this thread's psi element: a warp covers 8 vectors x 4 columns = 32 distinct banks of a B image
    const int v = (lt & 7) | ((lt >> 2) & 8), qb = ((lt >> 3) & 3) | ((lt >> 6) << 2), k = P.k;
    const int n_units = P.B / T2_UNIT_COLS;
    const uint32_t chunk = (uint32_t)(p & 15) >> 1;
    const uint32_t m_row = (uint32_t)((p & 63) >> 4) * 8192u + (uint32_t)(p >> 6) * 4096u + (uint32_t)(p & 1) * 8u;
    uint32_t gt = 0;   // tiles of this group so far = units so far
    for (int item = blockIdx.x; item < P.n_items; item += gridDim.x) {
        const int pr = item / P.S, strip = item - pr * P.S;
        const int rb = P.pairs[P.pstride * pr], cb = P.pairs[P.pstride * pr + 1];
        const uint32_t i = (uint32_t)rb * P.B + strip * TC_TP + p;
        for (int u = 0; u < n_units; ++u, ++gt) {
            const int s2 = gt & 1;
            const uint32_t use = gt >> 1;
            const uint32_t j0 = (uint32_t)cb * P.B + (2 * u + g) * TC_TQ;
            const float2 x = (v < k && qb < TC_TQ) ? P.psi[(size_t)(j0 + qb) * k + v] : float2{0.f, 0.f};
            float2 ent[TC_NG][4], elo[TC_NG][4];   // (re, im) of the 8 entries and their low parts x - trunc(x)
#pragma unroll
            for (int gg = 0; gg < TC_NG; ++gg)
#pragma unroll
                for (int e = 0; e < 4; ++e) {
                    const uint32_t j = j0 + 4 * (gsel + 2 * gg) + e;
                    float hr, hi;
                    entry_upper<float>(P.G, nullptr, i, j, hr, hi);
                    ent[gg][e] = make_float2(hr, hi);
                    elo[gg][e] = make_float2(hr - __uint_as_float(__float_as_uint(hr) & 0xffffe000u),
                                             hi - __uint_as_float(__float_as_uint(hi) & 0xffffe000u));
                }
            if (use > 0) mbar_wait(&bar.mempty[s2], (use - 1) & 1);      // column-side MMAs of the unit two back are done
            unsigned char* ub = ubuf + s2 * T2_UNIT;
#pragma unroll
            for (int gg = 0; gg < TC_NG; ++gg)
#pragma unroll
                for (int e = 0; e < 4; ++e) {
                    const uint32_t c8 = 4u * gsel + e;
                    const uint32_t off = m_row + (uint32_t)(2 * g + gg) * 1024u + c8 * 128u + ((chunk ^ c8) << 4);
                    *reinterpret_cast<float2*>(ub + off) = ent[gg][e];
                    *reinterpret_cast<float2*>(ub + T2_IMG + off) = elo[gg][e];
                }
            // (the row side second: the MMAs of this group's previous tile finish during the stores above)
            if (gt > 0) mbar_wait(&bar.dempty[g], (gt - 1) & 1);   // the row-side MMAs of this group's previous tile are done
#pragma unroll
            for (int gg = 0; gg < TC_NG; ++gg) {
                const uint32_t ta = a_lane + (uint32_t)(T2_COL_ASTAGE + g * TC_A_STAGE_COLS + 8 * (gsel + 2 * gg));
                tmem_st4(ta, ent[gg][0].x, ent[gg][0].y, ent[gg][1].x, ent[gg][1].y);
                tmem_st4(ta + 4, ent[gg][2].x, ent[gg][2].y, ent[gg][3].x, ent[gg][3].y);
                tmem_st4(ta + 32, elo[gg][0].x, elo[gg][0].y, elo[gg][1].x, elo[gg][1].y);
                tmem_st4(ta + 36, elo[gg][2].x, elo[gg][2].y, elo[gg][3].x, elo[gg][3].y);
            }
            t2_psi_image(bimg + g * TC_STAGE, v, qb, x);
            asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
            asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
            __syncwarp();
            if (lane == 0) {
                mbar_arrive(&bar.dfull[g]);
                mbar_arrive(&bar.mfull[s2]);
            }
        }
    }
}

// Converter group g of the cached variant (256 threads): the unit's raw image has been landed by a bulk copy in the
// layout the generator threads write; a thread reads the same 8 entries it would have generated (tile 2u + g, row p,
// column groups gsel, gsel + 2), writes their low parts x - trunc(x) to the lo image and the four row-side images to
// TMEM.  The raw stage is freed by the column-side MMAs' commit, not by the converters.
__device__ __forceinline__ void t2_convert(const T2Params& P, unsigned char* rawbuf, unsigned char* lobuf, unsigned char* bimg, T2Bars& bar,
                                           uint32_t d_tmem)
{
    const int tid = threadIdx.x, lane = tid & 31;
    const int g = tid >> 8, lt = tid & 255;
    const int p = lt & (TC_TP - 1), gsel = lt >> 7;
    const uint32_t a_lane = d_tmem + ((uint32_t)(p & ~31) << 16);
    // (vector, column) of this thread's psi element: a warp covers 8 vectors x 4 columns = 32 distinct banks of a B image
    const int v = (lt & 7) | ((lt >> 2) & 8), qb = ((lt >> 3) & 3) | ((lt >> 6) << 2), k = P.k;
    const int n_units = P.B / T2_UNIT_COLS;
    const uint32_t chunk = (uint32_t)(p & 15) >> 1;
    const uint32_t m_row = (uint32_t)((p & 63) >> 4) * 8192u + (uint32_t)(p >> 6) * 4096u + (uint32_t)(p & 1) * 8u;
    uint32_t gt = 0;   // units so far
    for (int item = blockIdx.x; item < P.n_items; item += gridDim.x) {
        const int pr = item / P.S;
        const int cb = P.pairs[P.pstride * pr + 1];
        for (int u = 0; u < n_units; ++u, ++gt) {
            const int s2 = gt & 1, st = gt % T2C_STAGES;
            const uint32_t use = gt >> 1;
            const uint32_t j0 = (uint32_t)cb * P.B + (2 * u + g) * TC_TQ;
            const float2 x = (v < k && qb < TC_TQ) ? P.psi[(size_t)(j0 + qb) * k + v] : float2{0.f, 0.f};   // in flight during the wait
            mbar_wait(&bar.raw_full[st], (gt / T2C_STAGES) & 1);
            const unsigned char* raw = rawbuf + st * T2_IMG;
            float2 ent[TC_NG][4], elo[TC_NG][4];
            uint32_t off[TC_NG][4];
#pragma unroll
            for (int gg = 0; gg < TC_NG; ++gg)
#pragma unroll
                for (int e = 0; e < 4; ++e) {
                    const uint32_t c8 = 4u * gsel + e;
                    off[gg][e] = m_row + (uint32_t)(2 * g + gg) * 1024u + c8 * 128u + ((chunk ^ c8) << 4);
                    ent[gg][e] = *reinterpret_cast<const float2*>(raw + off[gg][e]);
                }
#pragma unroll
            for (int gg = 0; gg < TC_NG; ++gg)
#pragma unroll
                for (int e = 0; e < 4; ++e)
                    elo[gg][e] = make_float2(ent[gg][e].x - __uint_as_float(__float_as_uint(ent[gg][e].x) & 0xffffe000u),
                                             ent[gg][e].y - __uint_as_float(__float_as_uint(ent[gg][e].y) & 0xffffe000u));
            if (use > 0) mbar_wait(&bar.mempty[s2], (use - 1) & 1);   // the column-side MMAs of the unit two back are done
            unsigned char* lo = lobuf + s2 * T2_IMG;
#pragma unroll
            for (int gg = 0; gg < TC_NG; ++gg)
#pragma unroll
                for (int e = 0; e < 4; ++e) *reinterpret_cast<float2*>(lo + off[gg][e]) = elo[gg][e];
            if (gt > 0) mbar_wait(&bar.dempty[g], (gt - 1) & 1);      // the row-side MMAs of this group's previous tile are done
#pragma unroll
            for (int gg = 0; gg < TC_NG; ++gg) {
                const uint32_t ta = a_lane + (uint32_t)(T2_COL_ASTAGE + g * TC_A_STAGE_COLS + 8 * (gsel + 2 * gg));
                tmem_st4(ta, ent[gg][0].x, ent[gg][0].y, ent[gg][1].x, ent[gg][1].y);
                tmem_st4(ta + 4, ent[gg][2].x, ent[gg][2].y, ent[gg][3].x, ent[gg][3].y);
                tmem_st4(ta + 32, elo[gg][0].x, elo[gg][0].y, elo[gg][1].x, elo[gg][1].y);
                tmem_st4(ta + 36, elo[gg][2].x, elo[gg][2].y, elo[gg][3].x, elo[gg][3].y);
            }
            t2_psi_image(bimg + g * TC_STAGE, v, qb, x);
            asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
            asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
            __syncwarp();
            if (lane == 0) {
                mbar_arrive(&bar.dfull[g]);
                mbar_arrive(&bar.mfull[s2]);
            }
        }
    }
}

// Producer warp of the cached variant: one 32 KB bulk copy per unit into a ring of T2C_STAGES raw stages.
__device__ __forceinline__ void t2_produce(const T2Params& P, unsigned char* rawbuf, T2Bars& bar)
{
    const int n_units = P.B / T2_UNIT_COLS;
    uint32_t gt = 0;
    if (!elect_one()) return;
    for (int item = blockIdx.x; item < P.n_items; item += gridDim.x) {
        const int pr = item / P.S, strip = item - pr * P.S;
        const unsigned char* blk = reinterpret_cast<const unsigned char*>(P.cache) + (size_t)P.pairs[P.pstride * pr + 2] * P.B * P.B * 8 +
                                   (size_t)strip * n_units * T2_IMG;
        for (int u = 0; u < n_units; ++u, ++gt) {
            const int st = gt % T2C_STAGES;
            if (gt >= T2C_STAGES) mbar_wait(&bar.raw_empty[st], (gt / T2C_STAGES - 1) & 1);
            asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(&bar.raw_full[st])), "r"(T2_IMG) : "memory");
            asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(rawbuf + st * T2_IMG)),
                         "l"(blk + (size_t)u * T2_IMG), "r"(T2_IMG), "r"(smem_u32(&bar.raw_full[st]))
                         : "memory");
        }
    }
}

// Row-side MMA warp: the one-sided kernel's 8 MMAs per tile, tiles in column order (group = tile parity).
__device__ __forceinline__ void t2_row_mma(const T2Params& P, unsigned char* bimg, T2Bars& bar, uint32_t d_tmem)
{
    const int lane = threadIdx.x & 31;
    const int n_tiles = P.B / TC_TQ, n_units = P.B / T2_UNIT_COLS;
    uint32_t items_done = 0;
    for (int item = blockIdx.x; item < P.n_items; item += gridDim.x, ++items_done) {
        for (int t = 0; t < n_tiles; ++t) {
            const int g = t & 1;
            const uint32_t gt = items_done * n_units + (t >> 1);
            const int stg = g;
            mbar_wait(&bar.dfull[g], gt & 1);
            if (t == 0 && items_done > 0) mbar_wait(&bar.dacc_empty, (items_done - 1) & 1);   // the epilogue has read the accumulator
            asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
            if (elect_one()) {
                // interleaved layout: 4 K-steps of 8 k' = 4 columns x (re, im); A_hi x [B_hi | B_lo] (N = 64), A_lo x B_hi (N = 32)
                const uint64_t bd = umma_desc_sbo(smem_u32(bimg + stg * TC_STAGE), T2_BSBO);   // the start-address field takes plain additions
                const uint32_t a0 = d_tmem + (uint32_t)(T2_COL_ASTAGE + stg * TC_A_STAGE_COLS);
#pragma unroll
                for (int ks = 0; ks < 4; ++ks) {
                    const uint64_t b = bd + (uint64_t)((ks * 2 * TC_LBO) >> 4);
                    umma_tf32_ts<64>(d_tmem + T2_COL_DACC, a0 + 8 * ks, b, (t | ks) != 0);
                    umma_tf32_ts<32>(d_tmem + T2_COL_DACC, a0 + 32 + 8 * ks, b, 1);
                }
                umma_commit(&bar.dempty[g]);
                if (t == n_tiles - 1) umma_commit(&bar.ddone);
            }
            __syncwarp();
        }
    }
}

// Column-side MMA warp: per unit 16 K-steps x (raw image, lo image), A = the item's psi operand in TMEM.
// CACHED: the raw image is the TMA stage of the unit (freed by this warp's commit), the lo image one of two buffers.
template <bool CACHED>
__device__ __forceinline__ void t2_col_mma(const T2Params& P, unsigned char* ubuf, unsigned char* lobuf, T2Bars& bar, uint32_t d_tmem)
{
    const int lane = threadIdx.x & 31;
    const int n_units = P.B / T2_UNIT_COLS;
    uint32_t gu = 0, items_done = 0;
    for (int item = blockIdx.x; item < P.n_items; item += gridDim.x, ++items_done) {
        mbar_wait(&bar.psi_full, items_done & 1);
        for (int u = 0; u < n_units; ++u, ++gu) {
            const int ub = gu & 1;
            mbar_wait(&bar.mfull[ub], (gu >> 1) & 1);
            if (gu > 0) mbar_wait(&bar.macc_empty, (gu - 1) & 1);
            asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
            if (elect_one()) {
                const int st = gu % T2C_STAGES;
                const uint64_t bd_raw = umma_desc_sw128(smem_u32(CACHED ? ubuf + st * T2_IMG : ubuf + ub * T2_UNIT));
                const uint64_t bd_lo = CACHED ? umma_desc_sw128(smem_u32(lobuf + ub * T2_IMG)) : bd_raw + (uint64_t)(T2_IMG >> 4);
                const uint32_t a0 = d_tmem + (uint32_t)(T2_COL_PSI + 128 * (items_done & 1));
#pragma unroll
                for (int img = 0; img < 2; ++img)
#pragma unroll
                    for (int j = 0; j < 16; ++j) {
                        const uint64_t b = (img ? bd_lo : bd_raw) + (uint64_t)(((j >> 2) * 8192 + (j & 3) * 32) >> 4);
                        umma_tf32_ts<64>(d_tmem + T2_COL_MACC, a0 + 8 * j, b, (img | j) != 0);
                    }
                umma_commit(&bar.mempty[ub]);
                if (CACHED) umma_commit(&bar.raw_empty[st]);
                umma_commit(&bar.macc_full);
            }
            __syncwarp();
        }
    }
}

// Epilogue warps q = 0..3 (TMEM lanes 32q..): q = 2 (row half) + (0: hi image, 1: lo image); lane = op * 16 + v.
// They also build the psi operand of the NEXT item into the other TMEM buffer, a few rows per unit, so that neither
// MMA warp waits at an item boundary, and they free the row-side accumulator before they store what they read.
__device__ __forceinline__ void t2_epilogue(const T2Params& P, float* xch, T2Bars& bar, uint32_t d_tmem)
{
    const int tid = threadIdx.x, lane = tid & 31, q = (tid >> 5) - T2_W_EPI;
    const int h = q >> 1, lohi = q & 1, op = lane >> 4, v = lane & 15, k = P.k;
    const int n_units = P.B / T2_UNIT_COLS;
    const int per = (32 + n_units - 2) / (n_units - 1);   // row pairs of the next psi operand built per unit (n_units >= 4)
    const uint32_t lane_base = d_tmem + ((uint32_t)(32 * q) << 16);
    // row pairs [r2a, r2b) of the psi operand of `item` into buffer `buf`
    auto psi_rows = [&](int item, int buf, int r2a, int r2b) {
        const int pr = item / P.S, strip = item - pr * P.S;
        const float2* src = P.psi + ((size_t)P.pairs[P.pstride * pr] * P.B + (size_t)strip * TC_TP + 64 * h) * k + v;
#pragma unroll 4
        for (int r2 = r2a; r2 < r2b; ++r2) {
            float2 x0 = float2{0.f, 0.f}, x1 = float2{0.f, 0.f};
            if (v < k) {
                x0 = src[(size_t)(2 * r2) * k];
                x1 = src[(size_t)(2 * r2 + 1) * k];
            }
            float a0 = op ? x0.y : x0.x, a1 = op ? -x0.x : x0.y, a2 = op ? x1.y : x1.x, a3 = op ? -x1.x : x1.y;
            if (lohi) {
                a0 -= __uint_as_float(__float_as_uint(a0) & 0xffffe000u);
                a1 -= __uint_as_float(__float_as_uint(a1) & 0xffffe000u);
                a2 -= __uint_as_float(__float_as_uint(a2) & 0xffffe000u);
                a3 -= __uint_as_float(__float_as_uint(a3) & 0xffffe000u);
            }
            tmem_st4(lane_base + (uint32_t)(T2_COL_PSI + 128 * buf + 4 * r2), a0, a1, a2, a3);
        }
    };
    auto psi_publish = [&]() {
        asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
        asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
        __syncwarp();
        if (lane == 0) mbar_arrive(&bar.psi_full);
    };
    if ((int)blockIdx.x < P.n_items) {
        psi_rows(blockIdx.x, 0, 0, 32);
        psi_publish();
    }
    uint32_t gu = 0, items_done = 0;
    for (int item = blockIdx.x; item < P.n_items; item += gridDim.x, ++items_done) {
        const int pr = item / P.S, strip = item - pr * P.S;
        const int rb = P.pairs[P.pstride * pr], cb = P.pairs[P.pstride * pr + 1];
        const size_t row0 = (size_t)rb * P.B + (size_t)strip * TC_TP;
        const int next = item + gridDim.x;
        const float2* nsrc = nullptr;
        if (next < P.n_items) {
            const int npr = next / P.S, nstrip = next - npr * P.S;
            nsrc = P.psi + ((size_t)P.pairs[P.pstride * npr] * P.B + (size_t)nstrip * TC_TP + 64 * h) * k + v;
        }
        for (int u = 0; u < n_units; ++u, ++gu) {
            // rows of the next item's psi operand handled in this unit: loaded now, in flight during the wait
            const bool pipelined = per <= 2;
            const int r2a = u * per;
            float2 nx[4];
#pragma unroll
            for (int i = 0; i < 4; ++i) nx[i] = float2{0.f, 0.f};
            if (pipelined && nsrc && r2a < 32 && v < k) {
#pragma unroll
                for (int i = 0; i < 4; ++i)
                    if (2 * r2a + i < 64 && i < 2 * per) nx[i] = nsrc[(size_t)(2 * r2a + i) * k];
            }
            mbar_wait(&bar.macc_full, gu & 1);
            asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
            uint32_t r[32];
            tmem_ld32(lane_base + (uint32_t)(T2_COL_MACC + 32 * h), r);
            asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
            __syncwarp();
            if (lane == 0) mbar_arrive(&bar.macc_empty);
            // hand the quadrant piece to the sum warps: named barriers 1 + b (buffer b full) and 3 + b (buffer b read)
            const int xb = gu & 1;
            float* X = xch + xb * (T2_XCH / 4);
            if (gu >= 2) asm volatile("bar.sync %0, 192;" ::"r"(3 + xb) : "memory");
#pragma unroll
            for (int c = 0; c < 32; ++c) X[(q * 32 + c) * 32 + (lane ^ ((c & 1) << 4))] = __uint_as_float(r[c]);   // odd columns swapped by halves: the sum warps read without bank conflicts
            asm volatile("bar.arrive %0, 192;" ::"r"(1 + xb) : "memory");
            // the column-side MMA warp has passed its wait for THIS item's operand (its unit 0 is complete), so the
            // next arrival on psi_full cannot overtake it; the other buffer's readers (previous item) are done
            if (next < P.n_items && r2a < 32) {
                const int buf = (items_done + 1) & 1;
                if (pipelined) {
#pragma unroll
                    for (int i = 0; i < 2; ++i) {
                        if (i >= per || r2a + i >= 32) break;
                        const float2 x0 = nx[2 * i], x1 = nx[2 * i + 1];
                        float a0 = op ? x0.y : x0.x, a1 = op ? -x0.x : x0.y, a2 = op ? x1.y : x1.x, a3 = op ? -x1.x : x1.y;
                        if (lohi) {
                            a0 -= __uint_as_float(__float_as_uint(a0) & 0xffffe000u);
                            a1 -= __uint_as_float(__float_as_uint(a1) & 0xffffe000u);
                            a2 -= __uint_as_float(__float_as_uint(a2) & 0xffffe000u);
                            a3 -= __uint_as_float(__float_as_uint(a3) & 0xffffe000u);
                        }
                        tmem_st4(lane_base + (uint32_t)(T2_COL_PSI + 128 * buf + 4 * (r2a + i)), a0, a1, a2, a3);
                    }
                } else {
                    psi_rows(next, buf, r2a, min(32, r2a + per));
                }
                if (r2a + per >= 32) psi_publish();
            }
        }
        mbar_wait(&bar.ddone, items_done & 1);
        float acc[32];
        tc_epilogue_load(d_tmem + T2_COL_DACC, q, acc);
        asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
        __syncwarp();
        if (lane == 0) mbar_arrive(&bar.dacc_empty);   // the next item's row-side MMAs may start
        tc_epilogue_store(acc, P.work + ((size_t)(P.slot_multi + cb) * P.D + row0 + 32 * q + lane) * k, k);
    }
}

// Sum warps (64 threads): out[c][v] = sum over the four quadrant pieces (row halves x hi/lo images), thread = (v, c % 4).
__device__ __forceinline__ void t2_col_sums(const T2Params& P, const float* xch)
{
    const int et = threadIdx.x - 32 * T2_W_SUM, vv = et & 15, cc = et >> 4, k = P.k;
    const int n_units = P.B / T2_UNIT_COLS;
    uint32_t gu = 0;
    for (int item = blockIdx.x; item < P.n_items; item += gridDim.x) {
        const int pr = item / P.S, strip = item - pr * P.S;
        const int rb = P.pairs[P.pstride * pr], cb = P.pairs[P.pstride * pr + 1];
        float2* out_col = P.work + ((size_t)(P.slot_mcol0 + rb * P.S + strip) * P.D + (size_t)cb * P.B) * k;
        for (int u = 0; u < n_units; ++u, ++gu) {
            const int xb = gu & 1;
            const float* X = xch + xb * (T2_XCH / 4);
            asm volatile("bar.sync %0, 192;" ::"r"(1 + xb) : "memory");
            float re[8], im[8];
#pragma unroll
            for (int i8 = 0; i8 < 8; ++i8) {
                const int c = cc + 4 * i8;
                re[i8] = im[i8] = 0.f;
#pragma unroll
                for (int qq = 0; qq < 4; ++qq) {
                    re[i8] += X[(qq * 32 + c) * 32 + (vv ^ ((c & 1) << 4))];
                    im[i8] += X[(qq * 32 + c) * 32 + ((16 + vv) ^ ((c & 1) << 4))];
                }
            }
            asm volatile("bar.arrive %0, 192;" ::"r"(3 + xb) : "memory");   // the buffer may be overwritten
#pragma unroll
            for (int i8 = 0; i8 < 8; ++i8)
                if (vv < k) out_col[(size_t)(u * T2_UNIT_COLS + cc + 4 * i8) * k + vv] = make_float2(re[i8], im[i8]);
        }
    }
}

template <bool CACHED>
__global__ void __launch_bounds__(CACHED ? T2C_THREADS : T2_THREADS, 1) pairs_tc_kernel(const T2Params P)
{
    extern __shared__ __align__(128) unsigned char smem_raw2_[];
    __shared__ __align__(8) T2Bars bar;
    __shared__ uint32_t s_tmem;
    const int tid = threadIdx.x, w = tid >> 5;
    // 1 KB aligned (128-byte swizzle atoms).  Generated: [unit buffers: raw + lo images][B images][exchange];
    // cached: [raw stages][lo buffers][B images][exchange]
    unsigned char* ubuf = smem_raw2_ + ((1024u - (smem_u32(smem_raw2_) & 1023u)) & 1023u);
    unsigned char* lobuf = ubuf + T2C_STAGES * T2_IMG;                       // cached variant only
    unsigned char* bimg = CACHED ? lobuf + 2 * T2_IMG : ubuf + 2 * T2_UNIT;
    float* xch = reinterpret_cast<float*>(bimg + 2 * TC_STAGE);
    if (tid == 0) {
        for (int g = 0; g < 2; ++g) {
            mbar_init(&bar.dfull[g], T2_GEN_WARPS / 2);
            mbar_init(&bar.dempty[g], 1);
        }
        for (int s = 0; s < 2; ++s) {
            mbar_init(&bar.mfull[s], T2_GEN_WARPS);
            mbar_init(&bar.mempty[s], 1);
        }
        for (int s = 0; s < T2C_STAGES; ++s) {
            mbar_init(&bar.raw_full[s], 1);
            mbar_init(&bar.raw_empty[s], 1);
        }
        mbar_init(&bar.macc_full, 1);
        mbar_init(&bar.macc_empty, 4);
        mbar_init(&bar.psi_full, 4);
        mbar_init(&bar.ddone, 1);
        mbar_init(&bar.dacc_empty, 4);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (w == T2_W_DMMA) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&s_tmem)), "n"(512) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const uint32_t d_tmem = s_tmem;

    if (w < T2_GEN_WARPS) {
        if (CACHED) t2_convert(P, ubuf, lobuf, bimg, bar, d_tmem);
        else t2_generate(P, ubuf, bimg, bar, d_tmem);
    } else if (w < T2_W_EPI + 4) t2_epilogue(P, xch, bar, d_tmem);
    else if (w < T2_W_SUM + 2) t2_col_sums(P, xch);
    else if (w == T2_W_DMMA) t2_row_mma(P, bimg, bar, d_tmem);
    else if (w == T2_W_MMMA) t2_col_mma<CACHED>(P, ubuf, lobuf, bar, d_tmem);
    else if (CACHED && w == T2C_W_TMA) t2_produce(P, ubuf, bar);

    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if (w == T2_W_DMMA) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(d_tmem), "n"(512) : "memory");
}

bool tc_pairs_supported(int dtype, int k, int B)
{
    return dtype == MFH_C64 && k > 1 && k <= 16 && B % TC_TP == 0;
}

static void t2_common_params(mfh_handle h, const void* psi, T2Params& P)
{
    const Plan& p = h->plan;
    P.G.K = make_philox_keys(h->seed);
    P.G.gc.neg_k2_ln2 = (float)(-0.6931471805599453 / (double)h->D);
    P.G.tab_global = nullptr;
    P.B = p.B;
    P.n_blk = p.n_blk;
    P.k = p.k;
    P.slot_multi = p.slot_multi;
    P.slot_mcol0 = p.slot_mcol0;
    P.S = p.B / TC_TP;
    P.D = h->D;
    P.cache = (const float2*)h->d_cache;
    P.psi = (const float2*)psi;
    P.work = (float2*)h->d_work;
}

// Generated block pairs: both positions from one generation.
static int launch_proc_pairs_tc(mfh_handle h, const void* psi, cudaStream_t st)
{
    T2Params P;
    t2_common_params(h, psi, P);
    P.pstride = 2;
    P.pairs = h->d_tc_pairs;
    P.n_items = (int32_t)(h->plan.tc_pairs.size() / 2) * P.S;
    if (int rc = ensure_dyn_smem(h, pairs_tc_kernel<false>, T2_SMEM)) return rc;
    pairs_tc_kernel<false><<<std::min(P.n_items, h->sm_count), T2_THREADS, T2_SMEM, st>>>(P);
    MFH_CUDA_CHECK(cudaGetLastError());
    return MFH_OK;
}

// Stored pair blocks (complex64 k-vector pair cache): both positions from ONE read of the stored block.
int launch_cached_pairs_tc(mfh_handle h, const void* psi, cudaStream_t st)
{
    T2Params P;
    t2_common_params(h, psi, P);
    P.pstride = 3;
    P.pairs = h->d_tc_cpairs;
    P.n_items = (int32_t)(h->plan.tc_cpairs.size() / 3) * P.S;
    if (P.n_items == 0) return MFH_OK;
    if (int rc = ensure_dyn_smem(h, pairs_tc_kernel<true>, T2C_SMEM)) return rc;
    pairs_tc_kernel<true><<<std::min(P.n_items, h->sm_count), T2C_THREADS, T2C_SMEM, st>>>(P);
    MFH_CUDA_CHECK(cudaGetLastError());
    return MFH_OK;
}

bool tc_multi_supported(mfh_handle h)
{
    // seeded source only: the generator warps of this kernel are the Philox / SFU Box-Muller path
    return h->kind != MFH_SRC_ANALYTIC && h->dtype == MFH_C64 && h->plan.k > 1 && h->plan.k <= 16 && h->plan.B % TC_TP == 0;
}

int launch_proc_multi_tc(mfh_handle h, const void* psi, cudaStream_t st)
{
    const Plan& p = h->plan;
    TcParams P;
    P.G.K = make_philox_keys(h->seed);
    P.G.gc.neg_k2_ln2 = (float)(-0.6931471805599453 / (double)h->D);
    P.G.tab_global = nullptr;
    P.B = p.B;
    P.n_blk = p.n_blk;
    P.k = p.k;
    P.slot_multi = p.slot_multi;
    P.D = h->D;
    P.cache_slot = h->d_cache_slot;
    P.skip = p.tc_pairs.empty() ? nullptr : h->d_tc_skip;
    P.pos = p.tc_left.empty() ? nullptr : h->d_tc_left;
    P.psi = (const float2*)psi;
    P.work = (float2*)h->d_work;
    if (!p.tc_pairs.empty())   // block pairs generated once for both sides
        if (int rc = launch_proc_pairs_tc(h, psi, st)) return rc;
    // what is left for the one-sided kernel: diagonal blocks and positions whose mirror image is cached
    if (p.owned_blocks - p.covered_blocks - (int64_t)p.tc_pairs.size() <= 0) return MFH_OK;
    const size_t smem = (size_t)TC_STAGES * TC_STAGE;
    if (int rc = ensure_dyn_smem(h, proc_multi_tc_kernel, (int)smem)) return rc;
    if (P.pos) proc_multi_tc_kernel<<<dim3((unsigned)(p.B / TC_TP), (unsigned)(p.tc_left.size() / 2)), TC_THREADS, smem, st>>>(P);
    else proc_multi_tc_kernel<<<dim3((unsigned)(h->D / TC_TP), p.n_blk), TC_THREADS, smem, st>>>(P);
    MFH_CUDA_CHECK(cudaGetLastError());
    return MFH_OK;
}

// --------------------------------------------------------------------------------------------
// Cached k-vector kernel (complex64): "reads each V block once for k vectors" (north_star (c);
// Y = A X with R simultaneous vectors, Eq. 12, on cached blocks P:177-183).
//
// A cached block is row-major B x B interleaved complex64, i.e. a real K-major matrix
// [B rows][2B floats] with K index k' = 2 q + c (c = 0 real, 1 imaginary part of column q), and
//     [Re Phi | Im Phi][p] = sum_k' A[p][k'] Bmat[k'][:],   Bmat[2q] = [Re Psi_q | Im Psi_q],
//                                                            Bmat[2q+1] = [-Im Psi_q | Re Psi_q].
// HBM-bound: 8 bytes per entry against 128 flop, which only the tensor cores sustain.  A CTA owns
// 128 rows x one cached block and walks it in tiles of 16 complex columns (32 floats = 128 B per
// row).  For k-vector plans the cache is stored TILED: each [128 rows x 32 floats] tile is one
// contiguous 16 KB run in HBM (full DRAM page locality; a row-major block would give 128-byte
// pieces 8 KB apart), rows XOR-swizzled in 16-byte chunks so that the shared-memory image is read
// without bank conflicts.  A producer lane issues one TMA bulk copy (cp.async.bulk, 16 KB) per tile
// into a 4-stage shared-memory ring; 8 converter warps read their row's words, split them into TF32 hi + lo and write them with tcgen05.st into TMEM
// as the A operand, and build the psi images; the MMA warp issues 8 tcgen05.mma per tile (3xTF32:
// A_hi B_hi + A_hi B_lo + A_lo B_hi) and commits onto the mbarrier that frees the TMEM stage.
// --------------------------------------------------------------------------------------------
constexpr int CT_STAGES = 4;                  // shared-memory stages of raw tiles (TMA)
constexpr int CT_TSTAGES = 3;                 // TMEM stages of split A operands
constexpr int CT_KF = 32;                     // floats per tile row = 16 complex columns = 4 MMA K-steps
constexpr int CT_RAW = TC_TP * CT_KF * 4;     // 16 KB raw tile
constexpr int CT_B_TILE = TC_N * CT_KF * 4;   // 4 KB psi image
constexpr int CT_BSTAGE = 2 * CT_B_TILE;      // hi, lo
constexpr int CT_SBO = (CT_KF / 4) * 128;     // 1 KB between 8-column groups of a psi image
constexpr int CT_A_STAGE_COLS = 2 * CT_KF;    // A_hi, A_lo: 32 TMEM columns each
constexpr int CT_THREADS = 32 * (TC_GEN_WARPS + 2);   // 8 converter warps, MMA warp, TMA warp
constexpr int CT_PSI = (CT_KF / 2) * 16 * 8;  // psi rows of one tile: 16 columns x <= 16 vectors x 8 B
constexpr int CT_SMEM = CT_STAGES * (CT_RAW + CT_PSI) + CT_TSTAGES * CT_BSTAGE + 1024;   // + alignment slack

struct CtParams {
    int32_t B, n_blk, k, slot_multi;
    int64_t D;
    const int32_t* cache_slot;
    const uint8_t* skip;   // positions served by the two-sided cached kernel (nullptr: none)
    const int32_t* pos;    // compact list of the (row block, column block) positions to run (blockIdx.y), or nullptr: all
    const float2* cache;   // tiled layout
    const float2* psi;
    float2* work;
};

__global__ void __launch_bounds__(CT_THREADS, 2) cached_multi_tc_kernel(const CtParams P)
{
    extern __shared__ __align__(128) unsigned char smem_raw_[];
    __shared__ __align__(8) uint64_t raw_full[CT_STAGES], raw_empty[CT_STAGES], a_full[CT_TSTAGES], a_empty[CT_TSTAGES], done;
    __shared__ uint32_t s_tmem;
    const int tid = threadIdx.x, w = tid >> 5, lane = tid & 31;
    const int m = P.pos ? P.pos[2 * blockIdx.y + 1] : (int)blockIdx.y;
    const uint32_t i_base = (P.pos ? (uint32_t)P.pos[2 * blockIdx.y] * P.B : 0u) + blockIdx.x * TC_TP;
    const int n = (int)(i_base / (uint32_t)P.B);
    if (P.skip && P.skip[n * P.n_blk + m]) return;   // both positions of a stored pair: pairs_tc_kernel<true>, from one read
    int32_t slot = P.cache_slot[n * P.n_blk + m];
    // Hermitian pair cache (MFH_MODE_PAIRS with k > 1) without the unit-image layout (no room for the column-side slots): position (n,m) marked -2 is served by the stored canonical block
    // C = H^[m,n]: phi^[n] += C^dagger psi^[m].  The CTA's 128 output rows are 128 COLUMNS of C; it reads C a second
    // time, transposed (TR): a stage is 16 rows of C x those 128 columns = eight 2 KB pieces of eight neighbouring
    // tiles.  (This halves the MEMORY of a k-vector operator, not the bytes per apply: DESIGN.md 6.5.)
    const bool TR = (slot == -2);
    if (TR) slot = P.cache_slot[m * P.n_blk + n];
    if (slot < 0) return;   // generated block: the fused kernel's
    // 1024-byte aligned stage base (128B swizzle pattern repeats every 8 rows x 128 B)
    unsigned char* smem = smem_raw_ + ((1024u - (smem_u32(smem_raw_) & 1023u)) & 1023u);
    unsigned char* psis = smem + CT_STAGES * CT_RAW;    // [CT_STAGES][16 columns][k] complex, filled by the producer
    unsigned char* bimg = psis + CT_STAGES * CT_PSI;

    if (tid == 0) {
        for (int s = 0; s < CT_STAGES; ++s) {
            mbar_init(&raw_full[s], 1);
            mbar_init(&raw_empty[s], TC_GEN_WARPS / 2);
        }
        for (int s = 0; s < CT_TSTAGES; ++s) {
            mbar_init(&a_full[s], TC_GEN_WARPS / 2);
            mbar_init(&a_empty[s], 1);
        }
        mbar_init(&done, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (w == TC_GEN_WARPS) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&s_tmem)),
                     "n"(256)
                     : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const uint32_t d_tmem = s_tmem;
    const int n_tiles = P.B / (CT_KF / 2);
    // the strip's tiles: block slot, row tile (i_base - n B) / 128, then B/16 tiles of 16 KB
    const unsigned char* block = reinterpret_cast<const unsigned char*>(P.cache) + (size_t)slot * P.B * P.B * 8;
    const uint32_t rt_own = (i_base - (uint32_t)n * P.B) / TC_TP;   // the CTA's 128-row (TR: 128-column) tile index in its block
    const unsigned char* strip = block + (size_t)rt_own * (P.B / (CT_KF / 2)) * CT_RAW;

    if (w == TC_GEN_WARPS + 1) {
        // ---- TMA producer: lane 0 copies the tiles, lane 1 the psi rows.  Bulk copies issued by ONE thread are serviced
        // one after the other (~0.27 us each on B200); copies of different lanes overlap, so the two
        // copies of a stage come from two lanes. ----
        const uint32_t psi_bytes = (uint32_t)((CT_KF / 2) * P.k * sizeof(float2));
        for (int t = 0; t < n_tiles; ++t) {
            const int s = t % CT_STAGES, u = t / CT_STAGES;
            if (u > 0) mbar_wait(&raw_empty[s], (u - 1) & 1);
            if (lane == 0)
                asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(&raw_full[s])),
                             "r"(CT_RAW + psi_bytes)
                             : "memory");
            __syncwarp();
            if (TR) {
                // 16 rows of C (row tile t / 8, rows 16 (t % 8) ..) x the CTA's 128 columns: column tiles 8 rt_own .. + 7,
                // one 2 KB piece of each, issued by eight lanes
                if (lane >= 2 && lane < 10) {
                    const int j = lane - 2;
                    asm volatile(
                        "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                            smem_u32(smem + s * CT_RAW + j * 2048)),
                        "l"(block + ((size_t)(t >> 3) * (P.B / (CT_KF / 2)) + 8 * rt_own + j) * CT_RAW + (size_t)(t & 7) * 2048), "r"(2048),
                        "r"(smem_u32(&raw_full[s]))
                        : "memory");
                }
            }
            if (lane == 1) {
                // the 16 psi rows of the tile are contiguous in [D][k]: one 1-D bulk copy
                asm volatile(
                    "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                        smem_u32(psis + s * CT_PSI)),
                    "l"(P.psi + ((size_t)m * P.B + (size_t)t * (CT_KF / 2)) * P.k), "r"(psi_bytes), "r"(smem_u32(&raw_full[s]))
                    : "memory");
            } else if (lane == 0 && !TR) {
                // tile t of the strip: 16 KB contiguous in the tiled cache layout (mfh_internal.cuh tiled_cache_offset)
                asm volatile(
                    "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                        smem_u32(smem + s * CT_RAW)),
                    "l"(strip + (size_t)t * CT_RAW), "r"(CT_RAW), "r"(smem_u32(&raw_full[s]))
                    : "memory");
            }
        }
    } else if (w == TC_GEN_WARPS) {
        // ---- MMA warp ----
        for (int t = 0; t < n_tiles; ++t) {
            const int s = t % CT_TSTAGES, u = t / CT_TSTAGES;
            mbar_wait(&a_full[s], u & 1);
            asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
            if (elect_one()) {
                const uint32_t b0 = smem_u32(bimg + s * CT_BSTAGE);
                const uint32_t a0 = d_tmem + (uint32_t)(TC_ACC_COLS + s * CT_A_STAGE_COLS);
#pragma unroll
                for (int ks = 0; ks < CT_KF / 8; ++ks) {
                    const uint64_t b = umma_desc_sbo(b0 + ks * 2 * TC_LBO, CT_SBO);   // [B_hi | B_lo] / B_hi
                    umma_tf32_ts<64>(d_tmem, a0 + 8 * ks, b, (t | ks) != 0);
                    umma_tf32_ts<32>(d_tmem, a0 + CT_KF + 8 * ks, b, 1);
                }
                umma_commit(&a_empty[s]);
                if (t == n_tiles - 1) umma_commit(&done);
            }
            __syncwarp();
        }
    } else {
        // ---- converter warps: two groups of four warps take the tiles alternately (group g: tiles g, g + 2, ...), so
        // that the per-tile chain of a warp (wait, load, split, tcgen05.st, wait::st, fences, arrive) of one tile
        // overlaps with the other group's; thread = row p, all eight four-float groups of the row ----
        const int p = tid & (TC_TP - 1), grp = tid >> 7, k = P.k;
        const uint32_t a_lane = d_tmem + ((uint32_t)(p & ~31) << 16);
        const int v = p & 15, qb0 = p >> 4;      // psi elements (columns qb0 and qb0 + 8 of the tile, vector v)
        for (int t = grp; t < n_tiles; t += 2) {
            const int s = t % CT_STAGES, u = t / CT_STAGES;
            const int ts = t % CT_TSTAGES, tu = t / CT_TSTAGES;
            mbar_wait(&raw_full[s], u & 1);
            float2 x[2];
#pragma unroll
            for (int h2 = 0; h2 < 2; ++h2)
                x[h2] = (v < k) ? reinterpret_cast<const float2*>(psis + s * CT_PSI)[(qb0 + 8 * h2) * k + v] : float2{0.f, 0.f};
            float4 raw[8];
            if (!TR) {
                const unsigned char* rp = smem + s * CT_RAW + p * 128;
#pragma unroll
                for (int g = 0; g < 8; ++g) raw[g] = *reinterpret_cast<const float4*>(rp + ((g ^ (p & 7)) << 4));
            } else {
                const unsigned char* cp = smem + s * CT_RAW + (p >> 4) * 2048 + (p & 1) * 8;
                const int cc = (p & 15) >> 1;
#pragma unroll
                for (int g = 0; g < 8; ++g) {
                    const int a0 = 2 * g, a1 = a0 + 1;
                    const float2 e0 = *reinterpret_cast<const float2*>(cp + a0 * 128 + ((cc ^ (a0 & 7)) << 4));
                    const float2 e1 = *reinterpret_cast<const float2*>(cp + a1 * 128 + ((cc ^ (a1 & 7)) << 4));
                    raw[g] = make_float4(e0.x, e0.y, e1.x, e1.y);
                }
            }
            if (tu > 0) mbar_wait(&a_empty[ts], (tu - 1) & 1);
#pragma unroll
            for (int g = 0; g < 8; ++g) {
                const float l0 = raw[g].x - __uint_as_float(__float_as_uint(raw[g].x) & 0xffffe000u);
                const float l1 = raw[g].y - __uint_as_float(__float_as_uint(raw[g].y) & 0xffffe000u);
                const float l2 = raw[g].z - __uint_as_float(__float_as_uint(raw[g].z) & 0xffffe000u);
                const float l3 = raw[g].w - __uint_as_float(__float_as_uint(raw[g].w) & 0xffffe000u);
                const uint32_t ta = a_lane + (uint32_t)(TC_ACC_COLS + ts * CT_A_STAGE_COLS + 4 * g);
                tmem_st4(ta, raw[g].x, raw[g].y, raw[g].z, raw[g].w);
                tmem_st4(ta + CT_KF, l0, l1, l2, l3);
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(&raw_empty[s]);
            {
                float* b = reinterpret_cast<float*>(bimg + ts * CT_BSTAGE);
                constexpr int BT = CT_B_TILE / 4;
                const float sg = TR ? -1.f : 1.f;
#pragma unroll
                for (int h2 = 0; h2 < 2; ++h2) {
                    const int qb = qb0 + 8 * h2;
                    const int o_re = ((v & 7) * 16 + (v >> 3) * CT_SBO + (qb >> 1) * 128 + (qb & 1) * 8) / 4;
                    const int o_im = o_re + 2 * CT_SBO / 4;
                    float prh, prl, pih, pil;
                    split_tf32(x[h2].x, prh, prl);
                    split_tf32(x[h2].y, pih, pil);
                    *reinterpret_cast<float2*>(b + o_re) = make_float2(prh, -sg * pih);
                    *reinterpret_cast<float2*>(b + o_im) = make_float2(pih, sg * prh);
                    *reinterpret_cast<float2*>(b + BT + o_re) = make_float2(prl, -sg * pil);
                    *reinterpret_cast<float2*>(b + BT + o_im) = make_float2(pil, sg * prl);
                }
            }
            asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
            asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
            __syncwarp();
            if (lane == 0) mbar_arrive(&a_full[ts]);
        }
        if (w < 4) {
            mbar_wait(&done, 0);
            tc_epilogue(d_tmem, w, P.work + ((size_t)(P.slot_multi + m) * P.D + i_base + 32 * w + lane) * k, k);
        }
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if (w == TC_GEN_WARPS)
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(d_tmem), "n"(256) : "memory");
}

bool tc_cached_multi_supported(int dtype, int k, int B) { return dtype == MFH_C64 && k > 1 && k <= 16 && B % TC_TP == 0; }

int launch_cached_multi_tc(mfh_handle h, const void* psi, cudaStream_t st)
{
    const Plan& p = h->plan;
    CtParams P;
    P.B = p.B;
    P.n_blk = p.n_blk;
    P.k = p.k;
    P.slot_multi = p.slot_multi;
    P.D = h->D;
    P.cache_slot = h->d_cache_slot;
    P.skip = p.tc_cpairs.empty() ? nullptr : h->d_tc_skip;
    P.pos = p.ct_left.empty() ? nullptr : h->d_ct_left;
    P.cache = (const float2*)h->d_cache;
    P.psi = (const float2*)psi;
    P.work = (float2*)h->d_work;
    if (int rc = ensure_dyn_smem(h, cached_multi_tc_kernel, CT_SMEM)) return rc;
    if (P.pos) cached_multi_tc_kernel<<<dim3((unsigned)(p.B / TC_TP), (unsigned)(p.ct_left.size() / 2)), CT_THREADS, CT_SMEM, st>>>(P);
    else cached_multi_tc_kernel<<<dim3((unsigned)(h->D / TC_TP), p.n_blk), CT_THREADS, CT_SMEM, st>>>(P);
    MFH_CUDA_CHECK(cudaGetLastError());
    return launch_cached_pairs_tc(h, psi, st);   // stored off-diagonal pairs in the unit-image layout: both sides from one read
}

}  // namespace mfh

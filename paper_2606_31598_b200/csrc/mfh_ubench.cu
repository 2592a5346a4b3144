// mfh_ubench.cu -- instruction-mix ceilings of the fused generate-and-apply kernels, measured on
// the device the library runs on (DESIGN.md 6.2 "ALU roofline").
//
// The procedural path is bound by plain ALU pipes, not by HBM or tensor cores: per generated entry
// one Philox4x32-10 call (18 32x32->64 multiplies + 18 three-input xors), the Box-Muller
// transcendentals and the multiply-accumulates.  B200's 32x32->64 multiply issues at a quarter of
// the FP32 rate and shares dispatch with the FP64 pipe, which no data sheet states; so instead of
// deriving a peak from nominal unit counts the library times a synthetic kernel that issues the
// SAME counts of IMAD.WIDE / LOP3 / DFMA / MUFU / FFMA per unit as the real inner loops, with no
// memory traffic, no shuffles and 4 independent units in flight per thread.  units/s of that
// kernel is the ceiling bench.py reports the fused kernels against.
#include <algorithm>
#include "mfh_internal.cuh"

namespace mfh {

constexpr int UB_ITER = 1024, UB_CH = 4, UB_THREADS = 256, UB_CTAS_PER_SM = 4;

// One unit per chain and iteration: NW wide multiplies (+ NW xors), NL further ALU ops, ND dfma,
// NM mufu, NF ffma.
// REG3: the DFMA chain takes three register operands (x = fma(x, y, z)) instead of two immediates.
template <int NW, int NL, int ND, int NM, int NF, bool REG3 = false>
__global__ void __launch_bounds__(UB_THREADS) ubench_kernel(uint32_t* out, uint32_t seed)
{
    uint32_t a[UB_CH], c[UB_CH];
    double d[UB_CH], d2[UB_CH];
    float f[UB_CH];
#pragma unroll
    for (int q = 0; q < UB_CH; ++q) {
        a[q] = threadIdx.x * (2 * q + 3) + seed;
        c[q] = a[q] ^ (0x9e3779b9u * (q + 1));
        d[q] = 1.0 + 1e-9 * a[q];
        d2[q] = 0.5 + 1e-9 * c[q];
        f[q] = 1.0f + 1e-6f * q;
    }
    for (int it = 0; it < UB_ITER; ++it) {
#pragma unroll
        for (int q = 0; q < UB_CH; ++q) {
#pragma unroll
            for (int r = 0; r < NW / 2; ++r) {   // two multiplies and two xors: one Philox round
                uint32_t lo0, hi0, lo1, hi1;
                mul_m0(a[q], lo0, hi0);
                mul_m1(c[q], lo1, hi1);
                a[q] = hi1 ^ lo0 ^ 0x9E3779B9u;
                c[q] = hi0 ^ lo1 ^ 0xBB67AE85u;
            }
#pragma unroll
            for (int r = 0; r < NL; ++r) c[q] = (c[q] & 0x7fffffffu) ^ (a[q] | (0x10u << r));   // one LOP3 each
            if (ND > 0) {
                double x = d[q] + __hiloint2double(0x3e000000, (int)a[q]);
#pragma unroll
                for (int r = 0; r < ND - 1; ++r) x = REG3 ? fma(x, d2[q], d[q]) : fma(x, 0.99999999, 1e-9);
                d[q] = x;
            }
            if (NM + NF > 0) {
                float y = f[q] + __uint_as_float(0x30000000u | (c[q] >> 12));
#pragma unroll
                for (int r = 0; r < NM; ++r) asm volatile("ex2.approx.ftz.f32 %0, %0;" : "+f"(y));
#pragma unroll
                for (int r = 0; r < NF; ++r) y = fmaf(y, 0.999f, 0.001f);
                f[q] = y;
            }
        }
    }
    uint32_t r = 0;
#pragma unroll
    for (int q = 0; q < UB_CH; ++q) r ^= a[q] ^ c[q] ^ (uint32_t)d[q] ^ (uint32_t)d2[q] ^ __float_as_uint(f[q]);
    out[blockIdx.x * blockDim.x + threadIdx.x] = r;
}

template <int NW, int NL, int ND, int NM, int NF, bool REG3 = false>
static int run_mix(int sm_count, cudaStream_t st, double* units_per_s)
{
    const int grid = sm_count * UB_CTAS_PER_SM;
    uint32_t* out = nullptr;
    MFH_CUDA_CHECK(cudaMalloc(&out, (size_t)grid * UB_THREADS * sizeof(uint32_t)));
    cudaEvent_t e0, e1;
    if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) {
        cudaFree(out);
        set_error("pipe-rate microbenchmark: cudaEventCreate failed");
        return MFH_ERR_CUDA;
    }
    float best = 1e30f;
    for (int rep = 0; rep < 4; ++rep) {   // first repetition warms up
        cudaEventRecord(e0, st);
        ubench_kernel<NW, NL, ND, NM, NF, REG3><<<grid, UB_THREADS, 0, st>>>(out, (uint32_t)rep);
        cudaEventRecord(e1, st);
        cudaError_t e = cudaEventSynchronize(e1);
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        if (e != cudaSuccess || cudaGetLastError() != cudaSuccess) {
            cudaEventDestroy(e0);
            cudaEventDestroy(e1);
            cudaFree(out);
            set_error("pipe-rate microbenchmark failed: %s", cudaGetErrorString(e));
            return MFH_ERR_CUDA;
        }
        if (rep > 0) best = std::min(best, ms);
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(out);
    *units_per_s = (double)grid * UB_THREADS * UB_ITER * UB_CH / ((double)best * 1e-3);
    return MFH_OK;
}

// ---- component ceilings: the library's OWN device functions, one component at a time ----------
// The synthetic mixes above issue instruction counts typed in from the SASS; these kernels call the generator code
// of mfh_gen.cuh itself, in the fused kernel's shape (8 warps, 2 CTAs per SM, 4 rows per lane, one column per step),
// so they follow every change of the generator:
//   COMP_PHILOX      pair_words() for 4 rows x 1 column per step, words xor-reduced          -> pairs/s
//   COMP_PHILOX_BM   + Gen<T>::normals() (tables in shared memory as in the fused kernel), entries summed
//   COMP_MAC         the two-sided multiply-accumulate of the fused kernel (8 FMA per pair, psi_j from shared memory,
//                    the column accumulator rotated by two shuffles per step) on entries that cost half an add each
constexpr int CP_ITER = 256, CP_R = 4, CP_THREADS = 256, CP_CTAS = 2, CP_SUB = 32;

template <typename T, int COMP>
__global__ void __launch_bounds__(CP_THREADS, CP_CTAS) comp_kernel(const GenArgs<T> G, typename Cplx<T>::type* out)
{
    using CT = typename Cplx<T>::type;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const typename Gen<T>::Tab* tab = stage_gen_table<T>(G);
    CT* psiw = reinterpret_cast<CT*>(smem_raw) + (threadIdx.x >> 5) * 32;
    const int lane = threadIdx.x & 31;
    psiw[lane] = CT{T(1) / T(lane + 1), T(lane) * T(0.001)};
    __syncthreads();
    const uint32_t i0 = (blockIdx.x * CP_THREADS + threadIdx.x) * 7u;
    T accr[CP_R], acci[CP_R], cr = T(0), ci = T(0);
    CT psi_i[CP_R];
    uint32_t xacc = 0;
#pragma unroll
    for (int r = 0; r < CP_R; ++r) {
        accr[r] = acci[r] = T(0);
        psi_i[r] = CT{T(0.5) + T(r), T(0.25) - T(r)};
    }
    T er = T(1e-3) * T(lane), ei = T(2e-3);
    for (int sub = 0; sub < CP_ITER / CP_SUB; ++sub) {
        const uint32_t j0 = 0x40000000u + blockIdx.x * 4096u + sub * CP_SUB;
#pragma unroll 1
        for (int s = 0; s < CP_SUB; ++s) {
            const int c = (lane + s) & 31;
            const CT p = psiw[c];
            if (COMP == 2) { er += T(1e-6); ei -= T(1e-6); }
#pragma unroll
            for (int r = 0; r < CP_R; ++r) {
                T hr, hi;
                if (COMP == 0) {
                    uint32_t x0, x1;
                    pair_words(G.K, i0 + 32 * r, j0 + c, x0, x1);
                    xacc ^= x0 ^ (x1 >> 1);
                    continue;
                } else if (COMP == 1) {
                    entry_upper<T>(G, tab, i0 + 32 * r, j0 + c, hr, hi);
                    accr[r] += hr;
                    acci[r] += hi;
                    continue;
                } else {
                    hr = er;
                    hi = ei;
                }
                accr[r] = fma(hr, p.x, accr[r]);
                accr[r] = fma(-hi, p.y, accr[r]);
                acci[r] = fma(hr, p.y, acci[r]);
                acci[r] = fma(hi, p.x, acci[r]);
                cr = fma(hr, psi_i[r].x, cr);
                cr = fma(hi, psi_i[r].y, cr);
                ci = fma(hr, psi_i[r].y, ci);
                ci = fma(-hi, psi_i[r].x, ci);
            }
            if (COMP == 2) {
                cr = __shfl_sync(0xffffffffu, cr, (lane + 1) & 31);
                ci = __shfl_sync(0xffffffffu, ci, (lane + 1) & 31);
            }
        }
    }
    T sr = cr + T(xacc & 1u), si = ci;
#pragma unroll
    for (int r = 0; r < CP_R; ++r) {
        sr += accr[r];
        si += acci[r];
    }
    out[blockIdx.x * CP_THREADS + threadIdx.x] = CT{sr, si};
}

template <typename T, int COMP> static int run_comp(int sm_count, cudaStream_t st, double* pairs_per_s)
{
    using CT = typename Cplx<T>::type;
    const int grid = sm_count * CP_CTAS;
    GenHostD host;
    make_gen_table(65536, host);
    GenArgs<T> G;
    G.K = make_philox_keys(0x1234567ull);
    G.an = AnalyticArgs{0, 0, 1, 0, 0, 0, 0};
    void* d_tab = nullptr;
    if constexpr (sizeof(T) == 8) {
        MFH_CUDA_CHECK(cudaMalloc(&d_tab, sizeof(GenTabD)));
        if (cudaMemcpy(d_tab, &host.tab, sizeof(GenTabD), cudaMemcpyHostToDevice) != cudaSuccess) {
            cudaFree(d_tab);
            set_error("component microbenchmark: table upload failed");
            return MFH_ERR_CUDA;
        }
        G.gc = host.gc;
        G.tab_global = (const GenTabD*)d_tab;
    } else {
        G.gc.neg_k2_ln2 = (float)(-0.6931471805599453 / 65536.0);
        G.tab_global = nullptr;
    }
    CT* out = nullptr;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    const size_t smem = (CP_THREADS / 32) * 32 * sizeof(CT);
    cudaError_t e = cudaMalloc(&out, (size_t)grid * CP_THREADS * sizeof(CT));
    if (e == cudaSuccess) e = cudaEventCreate(&e0);
    if (e == cudaSuccess) e = cudaEventCreate(&e1);
    float best = 1e30f;
    for (int rep = 0; rep < 4 && e == cudaSuccess; ++rep) {   // first repetition warms up
        cudaEventRecord(e0, st);
        comp_kernel<T, COMP><<<grid, CP_THREADS, smem, st>>>(G, out);
        cudaEventRecord(e1, st);
        e = cudaEventSynchronize(e1);
        if (e == cudaSuccess) e = cudaGetLastError();
        float ms = 0.f;
        if (e == cudaSuccess) cudaEventElapsedTime(&ms, e0, e1);
        if (rep > 0) best = std::min(best, ms);
    }
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
    if (out) cudaFree(out);
    if (d_tab) cudaFree(d_tab);
    if (e != cudaSuccess) {
        set_error("component microbenchmark failed: %s", cudaGetErrorString(e));
        return MFH_ERR_CUDA;
    }
    *pairs_per_s = (double)grid * CP_THREADS * CP_ITER * CP_R / ((double)best * 1e-3);
    return MFH_OK;
}

// Read-only HBM stream: every thread keeps 8 independent 128-bit non-allocating loads in flight over a
// grid-strided sweep of the buffer and xor-folds the words; one word per thread is written at the end.
// The denominator for kernels that READ a matrix once (a device-to-device copy, the MEASURED_PEAKS.json
// figure, also pays the write turn-around).
__global__ void __launch_bounds__(256) read_stream_kernel(const uint4* __restrict__ buf, size_t n16, uint32_t* out)
{
    uint32_t acc = 0;
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    for (; i + 7 * stride < n16; i += 8 * stride) {
        uint4 v[8];
#pragma unroll
        for (int u = 0; u < 8; ++u)
            asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0, %1, %2, %3}, [%4];"
                         : "=r"(v[u].x), "=r"(v[u].y), "=r"(v[u].z), "=r"(v[u].w)
                         : "l"(buf + i + u * stride));
#pragma unroll
        for (int u = 0; u < 8; ++u) acc ^= v[u].x ^ v[u].y ^ v[u].z ^ v[u].w;
    }
    for (; i < n16; i += stride) {
        const uint4 v = buf[i];
        acc ^= v.x ^ v.y ^ v.z ^ v.w;
    }
    out[blockIdx.x * blockDim.x + threadIdx.x] = acc;
}

}  // namespace mfh

using namespace mfh;

extern "C" MFH_API int mfh_debug_read_bandwidth(const void* buf_dev, size_t bytes, double* bytes_per_s, void* stream)
{
    if (!buf_dev || !bytes_per_s || bytes < (1u << 20) || ((uintptr_t)buf_dev & 15)) {
        set_error("mfh_debug_read_bandwidth: need a 16-byte aligned device buffer of at least 1 MiB");
        return MFH_ERR_INVALID_ARG;
    }
    int dev = 0, sms = 0;
    MFH_CUDA_CHECK(cudaGetDevice(&dev));
    MFH_CUDA_CHECK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    cudaStream_t st = (cudaStream_t)stream;
    const int grid = sms * 8;
    uint32_t* out = nullptr;
    MFH_CUDA_CHECK(cudaMalloc(&out, (size_t)grid * 256 * sizeof(uint32_t)));
    cudaEvent_t e0, e1;
    if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) {
        cudaFree(out);
        set_error("mfh_debug_read_bandwidth: cudaEventCreate failed");
        return MFH_ERR_CUDA;
    }
    float best = 1e30f;
    cudaError_t e = cudaSuccess;
    for (int rep = 0; rep < 4 && e == cudaSuccess; ++rep) {   // first repetition warms up
        cudaEventRecord(e0, st);
        read_stream_kernel<<<grid, 256, 0, st>>>((const uint4*)buf_dev, bytes / 16, out);
        cudaEventRecord(e1, st);
        e = cudaEventSynchronize(e1);
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        if (rep > 0) best = std::min(best, ms);
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(out);
    MFH_CUDA_CHECK(e);
    MFH_CUDA_CHECK(cudaGetLastError());
    *bytes_per_s = (double)(bytes / 16 * 16) / ((double)best * 1e-3);
    return MFH_OK;
}

// ---- complex multiply-accumulate streams in FP64 (the k-vector kernel of mfh_cached.cu) ----------------
// Measured on B200: a DFMA issues every 2 clocks only if one of its three 64-bit register operands comes from the
// operand reuse cache (the previous instruction of the same warp used the same register in the same slot); with
// three fresh registers it takes 3.  MS_REGS: the multiply-accumulate stream alone, psi values in registers, 32 DFMA
// per entry component in a row (every DFMA but the first reuses the entry) -- the ceiling of the pattern.  MS_LDS: the
// kernel's inner loop as written there (entry and psi values from shared memory every column, 8 vectors per thread):
// the compiler interleaves loads and DFMAs, fewer instructions hit the reuse cache -- the ceiling of the loop.
constexpr int MS_ITER = 4096, MS_KV = 8;
template <bool LDS>
__global__ void __launch_bounds__(256, 2) cmac_stream_kernel(double* out, const double* in)
{
    __shared__ __align__(16) double2 tile[128 * 17];
    __shared__ __align__(16) double2 ps[16 * 16];
    for (int i = threadIdx.x; i < 128 * 17; i += 256) tile[i] = make_double2(in[i % 60], in[(i + 7) % 60]);
    for (int i = threadIdx.x; i < 256; i += 256) ps[i] = make_double2(in[i % 64], in[(i + 3) % 64]);
    __syncthreads();
    const int row = threadIdx.x & 127, v0 = (threadIdx.x >> 7) * MS_KV;
    double ax[MS_KV], ay[MS_KV];
#pragma unroll
    for (int q = 0; q < MS_KV; ++q) ax[q] = ay[q] = 1e-9 * (threadIdx.x + q);
    if (LDS) {
        for (int it = 0; it < MS_ITER / 16; ++it) {
#pragma unroll 4
            for (int c = 0; c < 16; ++c) {
                const double2 hv = tile[row * 17 + c];
#pragma unroll
                for (int v = 0; v < MS_KV; ++v) {
                    const double2 p = ps[c * 16 + v0 + v];
                    ax[v] = fma(hv.x, p.x, ax[v]);
                    ax[v] = fma(-hv.y, p.y, ax[v]);
                    ay[v] = fma(hv.x, p.y, ay[v]);
                    ay[v] = fma(hv.y, p.x, ay[v]);
                }
            }
        }
    } else {
        double pr[MS_KV], pi[MS_KV];
#pragma unroll
        for (int q = 0; q < MS_KV; ++q) { pr[q] = ps[v0 + q].x; pi[q] = ps[v0 + q].y; }
        double hr = tile[row * 17].x, hi = tile[row * 17].y;
        for (int it = 0; it < MS_ITER; ++it) {
#pragma unroll
            for (int q = 0; q < MS_KV; ++q) { ax[q] = fma(hr, pr[q], ax[q]); ay[q] = fma(hr, pi[q], ay[q]); }
#pragma unroll
            for (int q = 0; q < MS_KV; ++q) { ax[q] = fma(-hi, pi[q], ax[q]); ay[q] = fma(hi, pr[q], ay[q]); }
            hr *= 0.999999;
            hi *= 1.000001;
        }
    }
    double s = 0.0;
#pragma unroll
    for (int q = 0; q < MS_KV; ++q) s += ax[q] + ay[q];
    out[blockIdx.x * 256 + threadIdx.x] = s;
}

// units = DFMA (thread instructions) per second
template <bool LDS> static int run_cmac_stream(int sm_count, cudaStream_t st, double* units_per_s)
{
    const int grid = sm_count * 2;
    double *out = nullptr, *in = nullptr;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    double host[64];
    for (int i = 0; i < 64; ++i) host[i] = 0.5 + 1e-3 * i;
    cudaError_t e = cudaMalloc(&out, (size_t)grid * 256 * sizeof(double));
    if (e == cudaSuccess) e = cudaMalloc(&in, sizeof host);
    if (e == cudaSuccess) e = cudaMemcpy(in, host, sizeof host, cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaEventCreate(&e0);
    if (e == cudaSuccess) e = cudaEventCreate(&e1);
    float best = 1e30f;
    for (int rep = 0; rep < 4 && e == cudaSuccess; ++rep) {   // first repetition warms up
        cudaEventRecord(e0, st);
        cmac_stream_kernel<LDS><<<grid, 256, 0, st>>>(out, in);
        cudaEventRecord(e1, st);
        e = cudaEventSynchronize(e1);
        float ms = 0.f;
        if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
        if (e == cudaSuccess) e = cudaGetLastError();
        if (rep > 0 && e == cudaSuccess) best = std::min(best, ms);
    }
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
    cudaFree(out);
    cudaFree(in);
    if (e != cudaSuccess) {
        set_error("FP64 multiply-accumulate stream microbenchmark failed: %s", cudaGetErrorString(e));
        return MFH_ERR_CUDA;
    }
    *units_per_s = (double)grid * 256 * MS_ITER * 4.0 * MS_KV / ((double)best * 1e-3);
    return MFH_OK;
}

extern "C" MFH_API int mfh_debug_pipe_rates(int32_t mix, double* units_per_s, void* stream)
{
    if (!units_per_s) { set_error("mfh_debug_pipe_rates: NULL pointer"); return MFH_ERR_INVALID_ARG; }
    if (mix < MFH_MIX_C128_PAIR || mix > MFH_PIPE_CMAC_LDS) {
        set_error("mfh_debug_pipe_rates: unknown mix %d", mix);
        return MFH_ERR_INVALID_ARG;
    }
    int dev = 0, sms = 0;
    MFH_CUDA_CHECK(cudaGetDevice(&dev));
    MFH_CUDA_CHECK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    cudaStream_t st = (cudaStream_t)stream;
    switch (mix) {
    // counts per unit from the SASS of the inner loops
    case MFH_MIX_C128_PAIR: return run_mix<14, 12, 32, 0, 0>(sms, st, units_per_s);
    case MFH_MIX_C64_ENTRY: return run_mix<14, 6, 0, 4, 11>(sms, st, units_per_s);
    case MFH_MIX_PHILOX: return run_mix<18, 0, 0, 0, 0>(sms, st, units_per_s);
    case MFH_MIX_DFMA31: return run_mix<0, 0, 32, 0, 0>(sms, st, units_per_s);
    case MFH_COMP_PHILOX: return run_comp<double, 0>(sms, st, units_per_s);
    case MFH_COMP_PHILOX_BM_C128: return run_comp<double, 1>(sms, st, units_per_s);
    case MFH_COMP_MAC_C128: return run_comp<double, 2>(sms, st, units_per_s);
    case MFH_COMP_PHILOX_BM_C64: return run_comp<float, 1>(sms, st, units_per_s);
    case MFH_COMP_MAC_C64: return run_comp<float, 2>(sms, st, units_per_s);
    // pipe model: which instruction classes overlap on sm_100
    case MFH_PIPE_WIDE16: return run_mix<16, 0, 0, 0, 0>(sms, st, units_per_s);
    case MFH_PIPE_LOP32: return run_mix<0, 32, 0, 0, 0>(sms, st, units_per_s);
    case MFH_PIPE_DFMA32: return run_mix<0, 0, 33, 0, 0>(sms, st, units_per_s);
    case MFH_PIPE_DFMA32_REG3: return run_mix<0, 0, 33, 0, 0, true>(sms, st, units_per_s);
    case MFH_PIPE_WIDE16_DFMA32: return run_mix<16, 0, 33, 0, 0>(sms, st, units_per_s);
    case MFH_PIPE_LOP32_DFMA32: return run_mix<0, 32, 33, 0, 0>(sms, st, units_per_s);
    case MFH_PIPE_WIDE16_LOP32: return run_mix<16, 32, 0, 0, 0>(sms, st, units_per_s);
    case MFH_PIPE_CMAC_REGS: return run_cmac_stream<false>(sms, st, units_per_s);
    case MFH_PIPE_CMAC_LDS: return run_cmac_stream<true>(sms, st, units_per_s);
    }
    set_error("mfh_debug_pipe_rates: unknown mix %d", mix);
    return MFH_ERR_INVALID_ARG;
}

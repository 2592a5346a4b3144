// mfh_sb.cu -- system-bath Hamiltonian action (NEXT-3):
//     H = H_S (x) I_B + I_S (x) H_B + g A (x) B_1   on   w in C^{d_S} (x) C^{d_B},
// the paper's own workload shape: two dense bath-side operators applied to R = d_S simultaneous
// state components (Eq. 12-13, n_op = 2).  With the state stored as X[b][s] (the library's k-vector
// layout [D][k], D = d_B, k = d_S):
//     Y = H_B X + g (B_1 X) A^T + X H_S^T.
// H_B and B_1 are two planned block operators of this library (cached blocks read once for the d_S
// columns by the tensor-core kernel of mfh_tc.cu, or generated); the O(d_B d_S^2) system-side mixing
// is one small kernel.  This file only composes: every O(d_B^2) step runs in the kernels above.
#include <algorithm>
#include <cmath>
#include <cstring>
#include <string>
#include <vector>
#include "mfh_internal.cuh"

struct mfh_sb_s {
    int64_t d_B = 0;
    int32_t d_S = 0, dtype = 0;
    double g = 0.0;
    mfh_handle hb = nullptr, b1 = nullptr;
    void* d_y1 = nullptr;      // H_B X
    void* d_y2 = nullptr;      // B_1 X
    double2* d_sys = nullptr;  // H_S then A, d_S x d_S complex doubles each, row-major
    std::vector<double> sys_host;   // the same on the host (uploaded by mfh_sb_plan)
    bool planned = false;
};

namespace mfh {

// out[b][s] = y1[b][s] + sum_s' ( H_S[s][s'] x[b][s'] + g A[s][s'] y2[b][s'] ); one thread per bath index b.
template <typename T>
__global__ void __launch_bounds__(256) sb_combine_kernel(int64_t d_B, int32_t k, double g, const double2* __restrict__ sys,
                                                         const typename Cplx<T>::type* __restrict__ x,
                                                         const typename Cplx<T>::type* __restrict__ y1,
                                                         const typename Cplx<T>::type* __restrict__ y2,
                                                         typename Cplx<T>::type* __restrict__ out)
{
    using CT = typename Cplx<T>::type;
    const double2* HS = sys;
    const double2* A = sys + k * k;
    for (int64_t b = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; b < d_B; b += (int64_t)gridDim.x * blockDim.x) {
        for (int s = 0; s < k; ++s) {
            const CT t = y1[b * k + s];
            double re = (double)t.x, im = (double)t.y;
            for (int sp = 0; sp < k; ++sp) {
                const CT xv = x[b * k + sp], yv = y2[b * k + sp];
                const double2 h = HS[s * k + sp], a = A[s * k + sp];
                re += h.x * (double)xv.x - h.y * (double)xv.y + g * (a.x * (double)yv.x - a.y * (double)yv.y);
                im += h.x * (double)xv.y + h.y * (double)xv.x + g * (a.x * (double)yv.y + a.y * (double)yv.x);
            }
            CT o;
            o.x = (T)re;
            o.y = (T)im;
            out[b * k + s] = o;
        }
    }
}

}  // namespace mfh

using namespace mfh;

extern "C" {

MFH_API int mfh_sb_create(mfh_sb_handle* out, int64_t d_B, int32_t d_S, int32_t B, uint64_t seed_HB, uint64_t seed_B1,
                          int32_t dtype, const double* HS_host, const double* A_host, double g)
{
    if (!out) { set_error("mfh_sb_create: out is NULL"); return MFH_ERR_INVALID_ARG; }
    *out = nullptr;
    if (d_S < 1 || d_S > MFH_MAX_K || !HS_host || !A_host || !std::isfinite(g)) {
        set_error("mfh_sb_create: need 1 <= d_S <= %d, H_S and A, finite g", MFH_MAX_K);
        return MFH_ERR_INVALID_ARG;
    }
    for (int s = 0; s < d_S; ++s)
        for (int t = 0; t < d_S; ++t) {   // both system-side matrices must be Hermitian
            const double* M[2] = {HS_host, A_host};
            for (const double* m : M)
                if (std::fabs(m[2 * (s * d_S + t)] - m[2 * (t * d_S + s)]) > 1e-12 * (1.0 + std::fabs(m[2 * (s * d_S + t)])) ||
                    std::fabs(m[2 * (s * d_S + t) + 1] + m[2 * (t * d_S + s) + 1]) > 1e-12 * (1.0 + std::fabs(m[2 * (s * d_S + t) + 1]))) {
                    set_error("mfh_sb_create: H_S and A must be Hermitian");
                    return MFH_ERR_INVALID_ARG;
                }
        }
    mfh_sb_handle h = new mfh_sb_s();
    int rc = mfh_create(&h->hb, d_B, B, seed_HB, MFH_SRC_GUE, 1.0, dtype, 0);
    if (!rc) rc = mfh_create(&h->b1, d_B, B, seed_B1, MFH_SRC_GUE, 1.0, dtype, 0);
    if (rc) {
        mfh_destroy(h->hb);
        mfh_destroy(h->b1);
        delete h;
        return rc;
    }
    h->d_B = d_B;
    h->d_S = d_S;
    h->dtype = dtype;
    h->g = g;
    // the system-side matrices travel to the device in mfh_sb_plan (no device work here)
    h->sys_host.assign(HS_host, HS_host + 2 * d_S * d_S);
    h->sys_host.insert(h->sys_host.end(), A_host, A_host + 2 * d_S * d_S);
    *out = h;
    return MFH_OK;
}

MFH_API int mfh_sb_destroy(mfh_sb_handle h)
{
    if (!h) return MFH_OK;
    mfh_destroy(h->hb);
    mfh_destroy(h->b1);
    if (h->d_y1) cudaFree(h->d_y1);
    if (h->d_y2) cudaFree(h->d_y2);
    if (h->d_sys) cudaFree(h->d_sys);
    delete h;
    return MFH_OK;
}

MFH_API int mfh_sb_plan(mfh_sb_handle h, int32_t mode, int64_t n_applies_hint, int64_t hbm_budget_bytes, void* stream,
                        char* json_out, size_t json_cap)
{
    if (!h) { set_error("mfh_sb_plan: NULL handle"); return MFH_ERR_INVALID_ARG; }
    if (h->planned) { set_error("mfh_sb_plan: already planned"); return MFH_ERR_BAD_STATE; }
    cudaStream_t st = (cudaStream_t)stream;
    const size_t vb = (size_t)h->d_B * h->d_S * complex_bytes(h->dtype);
    size_t free_b = 0, total_b = 0;
    MFH_CUDA_CHECK(cudaMemGetInfo(&free_b, &total_b));
    const double budget = (hbm_budget_bytes > 0 ? (double)hbm_budget_bytes : 0.9 * (double)free_b) - 2.0 * (double)vb;
    if (budget <= 0) { set_error("mfh_sb_plan: budget too small"); return MFH_ERR_OUT_OF_MEMORY; }
    char buf1[4096] = "", buf2[4096] = "";
    int rc = mfh_plan(h->hb, mode, h->d_S, n_applies_hint, (int64_t)(budget / 2), 0, stream, nullptr, 0);
    if (!rc) rc = mfh_plan(h->b1, mode, h->d_S, n_applies_hint, (int64_t)(budget / 2), 0, stream, nullptr, 0);
    if (rc) return rc;
    mfh_get_plan(h->hb, buf1, sizeof buf1);
    mfh_get_plan(h->b1, buf2, sizeof buf2);
    MFH_CUDA_CHECK(cudaMalloc(&h->d_y1, vb));
    MFH_CUDA_CHECK(cudaMalloc(&h->d_y2, vb));
    MFH_CUDA_CHECK(cudaMalloc(&h->d_sys, h->sys_host.size() * sizeof(double)));
    MFH_CUDA_CHECK(cudaMemcpy(h->d_sys, h->sys_host.data(), h->sys_host.size() * sizeof(double), cudaMemcpyHostToDevice));
    h->planned = true;
    MFH_CUDA_CHECK(cudaStreamSynchronize(st));
    if (json_out && json_cap) {
        std::string s = std::string("{\"d_B\":") + std::to_string(h->d_B) + ",\"d_S\":" + std::to_string(h->d_S) +
                        ",\"n_op\":2,\"flops_per_apply\":" + std::to_string(8.0 * 2.0 * (double)h->d_B * (double)h->d_B * h->d_S) +
                        ",\"H_B\":" + buf1 + ",\"B_1\":" + buf2 + "}";
        const size_t n = std::min(s.size(), json_cap - 1);
        memcpy(json_out, s.data(), n);
        json_out[n] = 0;
    }
    return MFH_OK;
}

MFH_API int mfh_sb_apply(mfh_sb_handle h, const void* x_dev, void* y_dev, void* stream)
{
    if (!h || !x_dev || !y_dev || x_dev == y_dev) { set_error("mfh_sb_apply: NULL or aliased pointer"); return MFH_ERR_INVALID_ARG; }
    if (!h->planned) { set_error("mfh_sb_apply: call mfh_sb_plan first"); return MFH_ERR_BAD_STATE; }
    cudaStream_t st = (cudaStream_t)stream;
    int rc = mfh_apply(h->hb, x_dev, h->d_y1, h->d_S, nullptr, stream);      // H_B X   (Eq. 12, R = d_S)
    if (!rc) rc = mfh_apply(h->b1, x_dev, h->d_y2, h->d_S, nullptr, stream);  // B_1 X
    if (rc) return rc;
    const int blocks = (int)std::min<int64_t>((h->d_B + 255) / 256, 148 * 8);
    if (h->dtype == MFH_C128)
        sb_combine_kernel<double><<<blocks, 256, 0, st>>>(h->d_B, h->d_S, h->g, h->d_sys, (const double2*)x_dev,
                                                           (const double2*)h->d_y1, (const double2*)h->d_y2, (double2*)y_dev);
    else
        sb_combine_kernel<float><<<blocks, 256, 0, st>>>(h->d_B, h->d_S, h->g, h->d_sys, (const float2*)x_dev,
                                                          (const float2*)h->d_y1, (const float2*)h->d_y2, (float2*)y_dev);
    MFH_CUDA_CHECK(cudaGetLastError());
    return MFH_OK;
}

}  // extern "C"

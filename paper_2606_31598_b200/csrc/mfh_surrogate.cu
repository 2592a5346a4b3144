// mfh_surrogate.cu -- neural surrogate of the planner (host code; Eq. 24-26, Algorithm 3).
//
// A one-hidden-layer network on componentwise normalised features predicts the logarithm of the measured apply
// time of a plan,   z = (x - mu) / sigma,   f(x) = tanh(z W1 + b1) W2 + b2   (Eq. 24),   t_NN = exp(f)   (Eq. 25),
// trained by minimising the log-time mean-squared error (Eq. 26) over benchmark records (x(p), t_mv(p)) that the
// measured planner (Algorithm 2) produces.  It only ranks candidates; a local measurement stays the decision rule.
// Parameter vector theta = [mu (F) | sigma (F) | W1 (F x H, row-major) | b1 (H) | W2 (H) | b2].
#include <cmath>
#include <cstring>
#include <vector>
#include "mfh_internal.cuh"

namespace mfh {

struct SurrView {
    int F, H;
    const double *mu, *sigma, *W1, *b1, *W2, *b2;
};
static SurrView view(const double* th, int F, int H)
{
    SurrView v{F, H, th, th + F, th + 2 * F, th + 2 * F + (size_t)F * H, th + 2 * F + (size_t)F * H + H,
               th + 2 * F + (size_t)F * H + 2 * H};
    return v;
}
static size_t theta_size(int F, int H) { return (size_t)2 * F + (size_t)F * H + 2 * (size_t)H + 1; }

// f(x) and, optionally, the hidden activations a = tanh(z W1 + b1) and z.
static double forward(const SurrView& v, const double* x, double* a_out, double* z_out)
{
    std::vector<double> z(v.F);
    for (int f = 0; f < v.F; ++f) z[f] = (x[f] - v.mu[f]) / v.sigma[f];
    double out = *v.b2;
    for (int h = 0; h < v.H; ++h) {
        double s = v.b1[h];
        for (int f = 0; f < v.F; ++f) s += z[f] * v.W1[(size_t)f * v.H + h];
        const double a = std::tanh(s);
        if (a_out) a_out[h] = a;
        out += a * v.W2[h];
    }
    if (z_out) memcpy(z_out, z.data(), v.F * sizeof(double));
    return out;
}

// Loss of Eq. 26 and its gradient with respect to [W1 | b1 | W2 | b2] (mu, sigma are data statistics, not trained).
static double loss_grad(const double* th, int F, int H, const double* X, const double* logt, int64_t n, double* grad)
{
    const SurrView v = view(th, F, H);
    const size_t np = (size_t)F * H + 2 * (size_t)H + 1;
    if (grad) std::fill(grad, grad + np, 0.0);
    std::vector<double> a(H), z(F);
    double loss = 0.0;
    for (int64_t i = 0; i < n; ++i) {
        const double r = forward(v, X + i * F, a.data(), z.data()) - logt[i];
        loss += r * r;
        if (!grad) continue;
        const double g = 2.0 * r / (double)n;
        double* gW1 = grad;
        double* gb1 = grad + (size_t)F * H;
        double* gW2 = gb1 + H;
        double* gb2 = gW2 + H;
        *gb2 += g;
        for (int h = 0; h < H; ++h) {
            gW2[h] += g * a[h];
            const double ds = g * v.W2[h] * (1.0 - a[h] * a[h]);
            gb1[h] += ds;
            for (int f = 0; f < F; ++f) gW1[(size_t)f * H + h] += ds * z[f];
        }
    }
    return loss / (double)n;
}

}  // namespace mfh

using namespace mfh;

extern "C" {

MFH_API int mfh_surrogate_features(int64_t D, int32_t dtype, int32_t k, int32_t mode, int32_t B, double flops_per_apply,
                                   double cache_bytes, double work_bytes, double free_bytes, int64_t n_task, int32_t p_row,
                                   int64_t waves, double gpu_bytes, int32_t sms, double* x_out)
{
    if (!x_out || D < 1 || B < 1 || k < 1 || n_task < 1 || p_row < 1 || waves < 1 || !(flops_per_apply > 0.0) ||
        !(free_bytes > 0.0) || !(gpu_bytes > 0.0) || sms < 1 || mode < MFH_MODE_PROCEDURAL || mode > MFH_MODE_PAIRS ||
        (dtype != MFH_C128 && dtype != MFH_C64)) {
        set_error("mfh_surrogate_features: invalid argument");
        return MFH_ERR_INVALID_ARG;
    }
    // x(p) of P:370, in the order of paper_2606_31598_b200/surrogate.py FEATURES
    double* x = x_out;
    x[0] = std::log((double)D);
    x[1] = std::log((double)k);
    x[2] = std::log((double)(D / B));
    x[3] = std::log((double)B);
    x[4] = std::log((double)n_task);
    x[5] = (double)p_row;
    x[6] = (double)waves;
    x[7] = mode == MFH_MODE_FULL;
    x[8] = mode == MFH_MODE_PARTIAL;
    x[9] = mode == MFH_MODE_PROCEDURAL;
    x[10] = mode == MFH_MODE_PAIRS;
    x[11] = std::log(flops_per_apply);
    x[12] = cache_bytes / free_bytes;
    x[13] = work_bytes / free_bytes;
    x[14] = (cache_bytes + work_bytes) / free_bytes;
    x[15] = dtype == MFH_C64;
    x[16] = std::log(gpu_bytes);
    x[17] = std::log((double)sms);
    return MFH_OK;
}

MFH_API int64_t mfh_surrogate_theta_size(int32_t n_features, int32_t hidden)
{
    if (n_features < 1 || hidden < 1) return 0;
    return (int64_t)theta_size(n_features, hidden);
}

MFH_API int mfh_surrogate_predict(const double* theta, int32_t n_features, int32_t hidden, const double* X, int64_t n,
                                  double* t_pred_seconds)
{
    if (!theta || !X || !t_pred_seconds || n_features < 1 || hidden < 1 || n < 0) {
        set_error("mfh_surrogate_predict: invalid argument");
        return MFH_ERR_INVALID_ARG;
    }
    const SurrView v = view(theta, n_features, hidden);
    for (int64_t i = 0; i < n; ++i) t_pred_seconds[i] = std::exp(forward(v, X + i * n_features, nullptr, nullptr));   // Eq. 25
    return MFH_OK;
}

MFH_API int mfh_surrogate_loss_grad(const double* theta, int32_t n_features, int32_t hidden, const double* X,
                                    const double* t_seconds, int64_t n, double* loss_out, double* grad_out)
{
    if (!theta || !X || !t_seconds || !loss_out || n_features < 1 || hidden < 1 || n < 1) {
        set_error("mfh_surrogate_loss_grad: invalid argument");
        return MFH_ERR_INVALID_ARG;
    }
    std::vector<double> logt(n);
    for (int64_t i = 0; i < n; ++i) {
        if (!(t_seconds[i] > 0.0)) { set_error("mfh_surrogate_loss_grad: times must be positive"); return MFH_ERR_INVALID_ARG; }
        logt[i] = std::log(t_seconds[i]);
    }
    *loss_out = loss_grad(theta, n_features, hidden, X, logt.data(), n, grad_out);
    return MFH_OK;
}

MFH_API int mfh_surrogate_fit(const double* X, const double* t_seconds, int64_t n, int32_t n_features, int32_t hidden,
                              int32_t epochs, double lr, uint64_t seed, double* theta_out, double* final_loss)
{
    if (!X || !t_seconds || !theta_out || n < 2 || n_features < 1 || hidden < 1 || epochs < 1 || !(lr > 0.0)) {
        set_error("mfh_surrogate_fit: invalid argument");
        return MFH_ERR_INVALID_ARG;
    }
    const int F = n_features, H = hidden;
    std::vector<double> logt(n);
    for (int64_t i = 0; i < n; ++i) {
        if (!(t_seconds[i] > 0.0) || !std::isfinite(t_seconds[i])) { set_error("mfh_surrogate_fit: times must be positive"); return MFH_ERR_INVALID_ARG; }
        logt[i] = std::log(t_seconds[i]);
    }
    double* mu = theta_out;
    double* sigma = theta_out + F;
    for (int f = 0; f < F; ++f) {   // componentwise normalisation; constant features get sigma = 1
        double m = 0.0, s2 = 0.0;
        for (int64_t i = 0; i < n; ++i) m += X[i * F + f];
        m /= (double)n;
        for (int64_t i = 0; i < n; ++i) s2 += (X[i * F + f] - m) * (X[i * F + f] - m);
        mu[f] = m;
        sigma[f] = s2 > 0.0 ? std::sqrt(s2 / (double)n) : 1.0;
    }
    const size_t np = (size_t)F * H + 2 * (size_t)H + 1;
    double* w = theta_out + 2 * F;
    uint64_t st = seed * 0x9E3779B97F4A7C15ull + 0xD1B54A32D192ED03ull;   // splitmix64 stream for the initial weights
    auto uni = [&]() {
        st += 0x9E3779B97F4A7C15ull;
        uint64_t zz = st;
        zz = (zz ^ (zz >> 30)) * 0xBF58476D1CE4E5B9ull;
        zz = (zz ^ (zz >> 27)) * 0x94D049BB133111EBull;
        zz ^= zz >> 31;
        return ((double)(zz >> 11) + 0.5) / 9007199254740992.0 * 2.0 - 1.0;
    };
    for (size_t q = 0; q < (size_t)F * H; ++q) w[q] = uni() / std::sqrt((double)F);
    for (int h = 0; h < H; ++h) w[(size_t)F * H + h] = 0.0;
    for (int h = 0; h < H; ++h) w[(size_t)F * H + H + h] = uni() / std::sqrt((double)H);
    double mean_y = 0.0;
    for (int64_t i = 0; i < n; ++i) mean_y += logt[i];
    w[np - 1] = mean_y / (double)n;
    // Adam on the full batch (the logs are a few thousand records at most)
    std::vector<double> g(np), m1(np, 0.0), m2(np, 0.0);
    const double b1 = 0.9, b2 = 0.999, eps = 1e-8;
    double loss = 0.0;
    for (int e = 1; e <= epochs; ++e) {
        loss = loss_grad(theta_out, F, H, X, logt.data(), n, g.data());
        const double c1 = 1.0 - std::pow(b1, e), c2 = 1.0 - std::pow(b2, e);
        for (size_t q = 0; q < np; ++q) {
            m1[q] = b1 * m1[q] + (1.0 - b1) * g[q];
            m2[q] = b2 * m2[q] + (1.0 - b2) * g[q] * g[q];
            w[q] -= lr * (m1[q] / c1) / (std::sqrt(m2[q] / c2) + eps);
        }
    }
    loss = loss_grad(theta_out, F, H, X, logt.data(), n, nullptr);
    if (final_loss) *final_loss = loss;
    return MFH_OK;
}

}  // extern "C"

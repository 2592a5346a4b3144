/*
 * mfh_oracle.c -- CPU ORACLE for phi = H psi.  TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A plain, slow, obviously-correct restatement of what the hot path computes, written
 * from the paper (/root/reference/PAPER.md, cited "P:<line>") and from the workload
 * definitions in BASELINE.json (configs[0..4]).  It shares no source, header, table or
 * constant generator with the CUDA path (paper_2606_31598_b200/csrc); neither imports the
 * other.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
 * reference legs may load this file's library.
 *
 * What is defined where
 *   - phi^[n] = sum_m H^[n,m] psi^[m]                      P:107-116 Eq. 4-5, Eq. 7
 *   - entries come from GLOBAL (i,j), never block labels
 *   - H^[m,n] = (H^[n,m])^dagger
 *   - Philox4x32-10 keyed on (seed, min(i,j), max(i,j)); Box-Muller; GUE normalisation
 *                                                          BASELINE.json configs[0]
 *   - H(lambda) = H0 + lambda V, H0 diagonal uniform       BASELINE.json configs[2]
 *   Readings where both are silent are listed in DESIGN.md ("Readings").
 *
 * Arithmetic: double for every entry, libm log/sqrt/cos/sin, long double accumulators,
 * built with -ffp-contract=off.  No blocking, fusion or reordering beyond the two-level
 * loop of Eq. 5/7.  OpenMP parallelism is over output rows only.
 *
 * Pins (tests/test_oracle_*.py): Philox known answers, closed-form uniforms, Box-Muller
 * identity and moments, bit-exact Hermiticity, explicit dense matmul at small D,
 * partition invariance, GUE moments / semicircle edge, <a|Hb> = conj<b|Ha>.
 * Parity unpinned against the paper (the paper fixes none of them):
 * the uniform mapping, the stream word of the counter, the H0 rule.
 */
#include <math.h>
#include <stdint.h>
#include <stddef.h>

/* ---- Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11), restated from its definition ---- */

#define ORC_PHILOX_M0 0xD2511F53u
#define ORC_PHILOX_M1 0xCD9E8D57u
#define ORC_PHILOX_W0 0x9E3779B9u
#define ORC_PHILOX_W1 0xBB67AE85u

void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        uint64_t p0 = (uint64_t)ORC_PHILOX_M0 * (uint64_t)c0;
        uint64_t p1 = (uint64_t)ORC_PHILOX_M1 * (uint64_t)c2;
        uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
        uint32_t n1 = (uint32_t)p1;
        uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
        uint32_t n3 = (uint32_t)p0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += ORC_PHILOX_W0;
        k1 += ORC_PHILOX_W1;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* Counter mapping (BASELINE.json configs[0]: "key=seed, counter=(i,j)"; R1):
 * key = (seed lo, seed hi); ctr = (min(i,j), max(i,j), stream, 0), 0-based global indices.
 * stream 0 = matrix entries, 1 = H0 diagonal. */
static void orc_words(uint64_t seed, uint32_t stream, uint32_t i, uint32_t j, uint32_t out[4])
{
    uint32_t key[2] = { (uint32_t)(seed & 0xffffffffu), (uint32_t)(seed >> 32) };
    uint32_t ctr[4] = { i < j ? i : j, i < j ? j : i, stream, 0u };
    orc_philox4x32_10(ctr, key, out);
}

void orc_philox_pairs(uint64_t seed, uint32_t stream, const uint32_t* i, const uint32_t* j,
                      int64_t n, uint32_t* words /* 4n */)
{
    for (int64_t t = 0; t < n; ++t) orc_words(seed, stream, i[t], j[t], words + 4 * t);
}

/* ---- uniforms and Box-Muller (R2, R3) ---- */

/* u = (x + 1/2) / 2^32: strictly inside (0,1), exact in double. */
double orc_uniform(uint32_t x) { return ((double)x + 0.5) * (1.0 / 4294967296.0); }

/* Basic (trigonometric) Box-Muller. */
void orc_box_muller(double u1, double u2, double* g1, double* g2)
{
    const double two_pi = 6.283185307179586;
    double r = sqrt(-2.0 * log(u1));
    *g1 = r * cos(two_pi * u2);
    *g2 = r * sin(two_pi * u2);
}

/* ---- entry rule (BASELINE.json configs[0]; Hermitian relation P:178-181) ----
 * i<j: (g1 + i g2)/sqrt(2D);  i>j: conjugate of entry (j,i);  i==j: g1/sqrt(D), real. */
void orc_entry(int64_t D, uint64_t seed, int64_t i, int64_t j, double* re, double* im)
{
    uint32_t w[4];
    double g1, g2;
    orc_words(seed, 0u, (uint32_t)i, (uint32_t)j, w);
    orc_box_muller(orc_uniform(w[0]), orc_uniform(w[1]), &g1, &g2);
    if (i == j) {
        *re = g1 / sqrt((double)D);
        *im = 0.0;
    } else {
        double s = 1.0 / sqrt(2.0 * (double)D);
        *re = g1 * s;
        *im = (i < j) ? g2 * s : -(g2 * s);
    }
}

/* Dense rectangle H[i0:i0+ni, j0:j0+nj], row-major interleaved (re,im). */
void orc_materialize(int64_t D, uint64_t seed, int64_t i0, int64_t ni, int64_t j0, int64_t nj,
                     double* out)
{
#pragma omp parallel for schedule(static)
    for (int64_t a = 0; a < ni; ++a)
        for (int64_t b = 0; b < nj; ++b)
            orc_entry(D, seed, i0 + a, j0 + b, out + 2 * (a * nj + b), out + 2 * (a * nj + b) + 1);
}

/* H0 diagonal of configs[2]: uniform in (-1,1); u from word 0 of ctr=(i,i,stream 1,0). */
void orc_h0(int64_t D, uint64_t seed_h0, double* h0)
{
    for (int64_t i = 0; i < D; ++i) {
        uint32_t w[4];
        orc_words(seed_h0, 1u, (uint32_t)i, (uint32_t)i, w);
        h0[i] = 2.0 * orc_uniform(w[0]) - 1.0;
    }
}

/* ---- blockwise H psi (Eq. 7), k simultaneous vectors (Eq. 12) ----
 * Psi, Phi_rows: row-major [row][k] interleaved complex.  rows == NULL means rows 0..nrows-1.
 * For global row i = n*B + alpha:  phi_i = sum_m sum_beta H(i, m*B+beta) psi_{m*B+beta}.
 * The entry is recomputed for every (i,j) it is needed at; nothing is cached. */
void orc_apply_rows(int64_t D, int64_t B, uint64_t seed, int64_t k, const double* Psi,
                    const int64_t* rows, int64_t nrows, double* Phi_rows)
{
    int64_t n_blk = D / B;
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t t = 0; t < nrows; ++t) {
        int64_t i = rows ? rows[t] : t;
        long double acc_re[64], acc_im[64]; /* k <= 64 */
        for (int64_t v = 0; v < k; ++v) { acc_re[v] = 0.0L; acc_im[v] = 0.0L; }
        for (int64_t m = 0; m < n_blk; ++m) {           /* input block m            */
            for (int64_t beta = 0; beta < B; ++beta) {  /* component inside block m */
                int64_t j = m * B + beta;
                double hr, hi;
                orc_entry(D, seed, i, j, &hr, &hi);
                for (int64_t v = 0; v < k; ++v) {
                    double pr = Psi[2 * (j * k + v)], pi = Psi[2 * (j * k + v) + 1];
                    acc_re[v] += (long double)hr * pr - (long double)hi * pi;
                    acc_im[v] += (long double)hr * pi + (long double)hi * pr;
                }
            }
        }
        for (int64_t v = 0; v < k; ++v) {
            Phi_rows[2 * (t * k + v)] = (double)acc_re[v];
            Phi_rows[2 * (t * k + v) + 1] = (double)acc_im[v];
        }
    }
}

/* Coupling scan of configs[2]: Phi[:,v] = h0 (.) Psi[:,v] + lambda_v (V Psi[:,v]),
 * V = GUE(seed_v), h0 from seed_h0.  Same row-subset convention as orc_apply_rows. */
void orc_apply_scan_rows(int64_t D, int64_t B, uint64_t seed_v, uint64_t seed_h0, int64_t k,
                         const double* lambdas, const double* Psi, const int64_t* rows,
                         int64_t nrows, double* Phi_rows)
{
    orc_apply_rows(D, B, seed_v, k, Psi, rows, nrows, Phi_rows);
    for (int64_t t = 0; t < nrows; ++t) {
        int64_t i = rows ? rows[t] : t;
        uint32_t w[4];
        orc_words(seed_h0, 1u, (uint32_t)i, (uint32_t)i, w);
        double h0 = 2.0 * orc_uniform(w[0]) - 1.0;
        for (int64_t v = 0; v < k; ++v) {
            double pr = Psi[2 * (i * k + v)], pi = Psi[2 * (i * k + v) + 1];
            Phi_rows[2 * (t * k + v)] = h0 * pr + lambdas[v] * Phi_rows[2 * (t * k + v)];
            Phi_rows[2 * (t * k + v) + 1] = h0 * pi + lambdas[v] * Phi_rows[2 * (t * k + v) + 1];
        }
    }
}

/* threads the OpenMP runtime will use (bench.py reports it as "cores") */
#ifdef _OPENMP
#include <omp.h>
int orc_num_threads(void) { return omp_get_max_threads(); }
#else
int orc_num_threads(void) { return 1; }
#endif

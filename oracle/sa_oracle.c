/*
 * sa_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, fp64 CPU statement of what the re-prefill hot path computes:
 * RoPE at absolute positions and causal softmax attention of new rows over a
 * logical (unpaged) context.  No pages, no tiles, no online softmax, no
 * splits, no blocking: the definition written out so it can be checked
 * against the paper by eye.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may call this.  It shares
 * no code, header, table or constant with paper_2607_00151_b200/csrc.
 *
 * Passages followed (PAPER.md line numbers):
 *   L311-313  "the i-th query token attends to prefix_j + i + 1 tokens",
 *             A_j = q_j*prefix_j + q_j(q_j+1)/2            -> mask, pair count
 *   L305      "a single query token that attends to its full KV cache of
 *             length L_j"                                   -> decode row = N=1
 *   L105-109  T(C) = T(S1) || ... || T(Sn)                  -> the context is
 *             the concatenation; a segment starts at absolute position P
 *   L422      grouped-query attention                       -> head h uses
 *             kv head floor(h/G)
 * RoPE (never mentioned in the paper; fixed by BASELINE.json and DESIGN.md
 * readings R1-R3): half-split pairing, theta_m = base^(-2m/D), no scaling.
 *
 * Parity pins: tests/test_oracle_pins.py (brute force, closed forms,
 * invariants, a library special case).  Absolute bf16 output values are
 * otherwise unpinned: the paper prints no tensor anywhere.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* Number of threads the parallel loops below will use (for reporting). */
int32_t sa_oracle_num_threads(void) {
#ifdef _OPENMP
    return (int32_t)omp_get_max_threads();
#else
    return 1;
#endif
}

/*
 * Step 1 (step 1).
 * x, out: [n, H, D] row-major doubles; pos[n] absolute positions.
 * For m in [0, D/2): theta_m = base^(-2m/D),
 *   out[m]       = x[m]      *cos(p*theta_m) - x[m+D/2]*sin(p*theta_m)
 *   out[m + D/2] = x[m + D/2]*cos(p*theta_m) + x[m]    *sin(p*theta_m)
 */
void sa_oracle_rope(const double *x, const int64_t *pos, int64_t n, int32_t H,
                    int32_t D, double base, double *out) {
    const int32_t half = D / 2;
#pragma omp parallel for schedule(static)
    for (int64_t t = 0; t < n; ++t) {
        const double p = (double)pos[t];
        for (int32_t h = 0; h < H; ++h) {
            const double *xi = x + ((size_t)t * H + h) * D;
            double *oi = out + ((size_t)t * H + h) * D;
            for (int32_t m = 0; m < half; ++m) {
                const double theta = pow(base, -2.0 * (double)m / (double)D);
                const double c = cos(p * theta), s = sin(p * theta);
                oi[m] = xi[m] * c - xi[m + half] * s;
                oi[m + half] = xi[m + half] * c + xi[m] * s;
            }
        }
    }
}

/*
 * Steps 2-4 for a list of (row, head) pairs.
 *   q  [N,  Hq,  D]  rotated queries of the new rows; row i sits at absolute
 *                    position P + i
 *   k  [L,  Hkv, D]  rotated keys of the whole logical context, L >= P + N
 *   v  [L,  Hkv, D]  values
 * For sample s = (i, h):  g = h / (Hq/Hkv);
 *   s_j   = sm_scale * sum_d q[i,h,d] * k[j,g,d]       for 0 <= j <= P + i
 *   m     = max_j s_j ;  Z = sum_j exp(s_j - m)
 *   o[s,:] = sum_j exp(s_j - m)/Z * v[j,g,:] ;  lse[s] = m + ln Z
 * Keys j > P + i are simply not in the sums.  rows == NULL means "every
 * (i, h)": sample s = i*Hq + h, n_samples must be N*Hq.
 * probs (nullable, tiny inputs only): [n_samples, L], p_j for j <= P+i, 0
 * elsewhere.  pair_count (nullable): number of (i, j) pairs visited, summed
 * over samples.
 */
void sa_oracle_attend(const double *q, const double *k, const double *v,
                      int64_t N, int64_t L, int32_t Hq, int32_t Hkv, int32_t D,
                      int64_t P, double sm_scale, int64_t n_samples,
                      const int64_t *rows, const int32_t *heads, double *o,
                      double *lse, double *probs, int64_t *pair_count) {
    const int32_t G = Hq / Hkv;
    int64_t pairs = 0;
    (void)N;
#pragma omp parallel for schedule(dynamic, 1) reduction(+ : pairs)
    for (int64_t s = 0; s < n_samples; ++s) {
        const int64_t i = rows ? rows[s] : s / Hq;
        const int32_t h = rows ? heads[s] : (int32_t)(s % Hq);
        const int32_t g = h / G;
        const int64_t n_keys = P + i + 1;
        const double *qi = q + ((size_t)i * Hq + h) * D;
        double *sc = (double *)malloc(sizeof(double) * (size_t)n_keys);
        double m = -INFINITY;
        for (int64_t j = 0; j < n_keys; ++j) {
            const double *kj = k + ((size_t)j * Hkv + g) * D;
            double dot = 0.0;
            for (int32_t d = 0; d < D; ++d) dot += qi[d] * kj[d];
            sc[j] = sm_scale * dot;
            if (sc[j] > m) m = sc[j];
        }
        double Z = 0.0;
        for (int64_t j = 0; j < n_keys; ++j) {
            sc[j] = exp(sc[j] - m);
            Z += sc[j];
        }
        double *os = o + (size_t)s * D;
        for (int32_t d = 0; d < D; ++d) os[d] = 0.0;
        for (int64_t j = 0; j < n_keys; ++j) {
            const double p = sc[j] / Z;
            const double *vj = v + ((size_t)j * Hkv + g) * D;
            for (int32_t d = 0; d < D; ++d) os[d] += p * vj[d];
            if (probs) probs[(size_t)s * L + j] = p;
        }
        if (probs)
            for (int64_t j = n_keys; j < L; ++j) probs[(size_t)s * L + j] = 0.0;
        lse[s] = m + log(Z);
        pairs += n_keys;
        free(sc);
    }
    if (pair_count) *pair_count = pairs;
}

// sa_scheduler.cu -- host core of the lookahead-aware request scheduler (
// PAPER.md section 4): the mixed-batch latency model of Eq. 1 (L349-353), its fit from
// sa_latency_table's measurements ("profiled coefficient", L309, L319), Algorithm 1 (slack-aware
// prefill batching, L321-347), Algorithm 2 (TBT-bounded hybrid batching, L363-388) and the sizing
// of a dynamic lookahead chunk (L59, L359, L396).  Plain host code: no device work.
//
// All estimates are evaluated in double precision in the order Eq. 1 is written:
//   c0 + T_GEMM(M) + alpha_d * sum_j L_j + alpha_p * sum_j A_j,
// with the integer sums M, sum L and sum A kept exactly (running sums replace the re-evaluation
// of the pseudo-code's EstBatchLatency(B + {c}); the value is the same bit for bit).
#include <math.h>

#include <cmath>

#include "sa_internal.h"

namespace {

struct Sums {
    int64_t n_dec = 0, tokens = 0;  // M = n_dec + tokens of prefill chunks (L301)
    int64_t sum_L = 0;              // L305-309
    int64_t sum_A = 0;              // L311-319
};

inline int64_t pairs(int64_t q, int64_t prefix) { return q * prefix + q * (q + 1) / 2; }  // L313

double t_gemm(const sa_latency_model *m, int64_t M) {
    const int n = m->n_gemm;
    if (n <= 0) return 0.0;
    const double x = double(M);
    if (n == 1 || x <= m->gemm_m[0]) return m->gemm_ms[0];
    for (int i = 0; i + 1 < n; ++i)
        if (x <= m->gemm_m[i + 1])
            return m->gemm_ms[i] + (x - m->gemm_m[i]) / (m->gemm_m[i + 1] - m->gemm_m[i]) * (m->gemm_ms[i + 1] - m->gemm_ms[i]);
    return m->gemm_ms[n - 1] +
           (x - m->gemm_m[n - 1]) / (m->gemm_m[n - 1] - m->gemm_m[n - 2]) * (m->gemm_ms[n - 1] - m->gemm_ms[n - 2]);
}

double est(const sa_latency_model *m, const Sums &s) {
    const int64_t M = s.n_dec + s.tokens;
    if (M == 0) return 0.0;
    return m->c0_ms + t_gemm(m, M) + m->alpha_d_ms * double(s.sum_L) + m->alpha_p_ms * double(s.sum_A);
}

bool model_ok(const sa_latency_model *m) {
    if (!m || m->n_gemm < 0 || m->n_gemm > SA_GEMM_TABLE_MAX) return false;
    for (int i = 0; i + 1 < m->n_gemm; ++i)
        if (!(m->gemm_m[i + 1] > m->gemm_m[i])) return false;
    return true;
}

bool chunks_ok(const sa_chunk *c, int32_t n) {
    if (n < 0 || (n > 0 && !c)) return false;
    for (int32_t i = 0; i < n; ++i)
        if (c[i].q < 0 || c[i].prefix < 0) return false;
    return true;
}

inline Sums with_decode(Sums s, int64_t L) {
    s.n_dec += 1;
    s.sum_L += L;
    return s;
}
inline Sums with_chunk(Sums s, const sa_chunk &c) {
    s.tokens += c.q;
    s.sum_A += pairs(c.q, c.prefix);
    return s;
}

// Solve the (at most 3 x 3) normal equations of a column-scaled least-squares problem by Gaussian
// elimination with partial pivoting.
bool solve(int n, double (*a)[4], double *x) {
    for (int c = 0; c < n; ++c) {
        int piv = c;
        for (int r = c + 1; r < n; ++r)
            if (fabs(a[r][c]) > fabs(a[piv][c])) piv = r;
        if (fabs(a[piv][c]) < 1e-300) return false;
        for (int k = 0; k <= n; ++k) {
            const double t = a[c][k];
            a[c][k] = a[piv][k];
            a[piv][k] = t;
        }
        for (int r = c + 1; r < n; ++r) {
            const double f = a[r][c] / a[c][c];
            for (int k = c; k <= n; ++k) a[r][k] -= f * a[c][k];
        }
    }
    for (int c = n - 1; c >= 0; --c) {
        double v = a[c][n];
        for (int k = c + 1; k < n; ++k) v -= a[c][k] * x[k];
        x[c] = v / a[c][c];
    }
    return true;
}

}  // namespace

extern "C" int32_t sa_est_batch_latency(const sa_latency_model *model, const int64_t *decode_L, int32_t n_dec,
                                        const sa_chunk *chunks, int32_t n_pre, double *out_ms) {
    if (!model_ok(model) || !out_ms || n_dec < 0 || (n_dec > 0 && !decode_L) || !chunks_ok(chunks, n_pre))
        return SA_ERR_INVALID_ARG;
    Sums s;
    for (int32_t i = 0; i < n_dec; ++i) {
        if (decode_L[i] < 0) return SA_ERR_INVALID_ARG;
        s = with_decode(s, decode_L[i]);
    }
    for (int32_t i = 0; i < n_pre; ++i) s = with_chunk(s, chunks[i]);
    *out_ms = est(model, s);
    return SA_OK;
}

extern "C" int32_t sa_schedule_hybrid(const sa_latency_model *model, const int64_t *decode_L, int32_t n_dec,
                                      const sa_chunk *lc, int32_t n_lc, const sa_chunk *be, int32_t n_be,
                                      double delta_ms, int32_t *out_admitted, double *out_est_ms) {
    if (!model_ok(model) || !out_admitted || n_dec < 0 || (n_dec > 0 && !decode_L) || !chunks_ok(lc, n_lc) ||
        !chunks_ok(be, n_be))
        return SA_ERR_INVALID_ARG;
    Sums s;
    int32_t a = 0, b = 0, c = 0;
    for (; a < n_dec; ++a) {  // Alg. 2 lines 3-6
        if (decode_L[a] < 0) return SA_ERR_INVALID_ARG;
        const Sums t = with_decode(s, decode_L[a]);
        if (est(model, t) > delta_ms) break;
        s = t;
    }
    for (; b < n_lc; ++b) {  // lines 8-11
        const Sums t = with_chunk(s, lc[b]);
        if (est(model, t) > delta_ms) break;
        s = t;
    }
    for (; c < n_be; ++c) {  // lines 13-16
        const Sums t = with_chunk(s, be[c]);
        if (est(model, t) > delta_ms) break;
        s = t;
    }
    out_admitted[0] = a;
    out_admitted[1] = b;
    out_admitted[2] = c;
    if (out_est_ms) *out_est_ms = est(model, s);
    return SA_OK;
}

extern "C" int32_t sa_schedule_prefill_slack(const sa_latency_model *model, const sa_lc_request *lc_queue, int32_t n_queue,
                                             double t_now_ms, const sa_chunk *lc_chunks, int32_t n_lc_chunks,
                                             const sa_chunk *be, int32_t n_be, int32_t *out_be_admitted,
                                             double *out_budget_ms, double *out_est_ms) {
    if (!model_ok(model) || !out_be_admitted || n_queue < 0 || (n_queue > 0 && !lc_queue) ||
        !chunks_ok(lc_chunks, n_lc_chunks) || !chunks_ok(be, n_be))
        return SA_ERR_INVALID_ARG;
    double p = 0.0, s_min = INFINITY;  // Alg. 1 line 4
    for (int32_t i = 0; i < n_queue; ++i) {  // lines 5-9
        const sa_lc_request &r = lc_queue[i];
        if (r.q < 0 || r.prefix < 0) return SA_ERR_INVALID_ARG;
        sa_chunk whole{r.q, r.prefix};
        p = p + est(model, with_chunk(Sums(), whole));  // EstPrefillLatency(r): the request's prefill alone
        const double s_j = (r.t_arrival_ms + r.slo_ttft_ms) - t_now_ms - p;
        s_min = fmin(s_min, s_j);
    }
    const double budget = fmax(0.0, s_min);  // line 10
    Sums s;
    for (int32_t i = 0; i < n_lc_chunks; ++i) s = with_chunk(s, lc_chunks[i]);  // line 12
    int32_t c = 0;
    for (; c < n_be; ++c) {  // lines 14-18: in order, stop at the first chunk that does not fit
        const Sums t = with_chunk(s, be[c]);
        if (est(model, t) > budget) break;
        s = t;
    }
    *out_be_admitted = c;
    if (out_budget_ms) *out_budget_ms = budget;
    if (out_est_ms) *out_est_ms = est(model, s);
    return SA_OK;
}

extern "C" int32_t sa_dynamic_chunk(const sa_latency_model *model, const int64_t *decode_L, int32_t n_dec,
                                    const sa_chunk *chunks, int32_t n_pre, int64_t prefix, int64_t remaining,
                                    int64_t max_chunk, int64_t granularity, double budget_ms, int64_t *out_q) {
    if (!model_ok(model) || !out_q || n_dec < 0 || (n_dec > 0 && !decode_L) || !chunks_ok(chunks, n_pre) || prefix < 0 ||
        remaining < 0 || max_chunk <= 0 || granularity <= 0)
        return SA_ERR_INVALID_ARG;
    Sums s;
    for (int32_t i = 0; i < n_dec; ++i) {
        if (decode_L[i] < 0) return SA_ERR_INVALID_ARG;
        s = with_decode(s, decode_L[i]);
    }
    for (int32_t i = 0; i < n_pre; ++i) s = with_chunk(s, chunks[i]);
    const int64_t top = remaining < max_chunk ? remaining : max_chunk;
    auto fits = [&](int64_t q) { return est(model, with_chunk(s, sa_chunk{q, prefix})) <= budget_ms; };
    *out_q = 0;
    if (top <= 0) return SA_OK;
    if (fits(top)) {
        *out_q = top;
        return SA_OK;
    }
    int64_t lo = 0, hi = (top - 1) / granularity;  // candidates k * granularity, k in [1, hi]
    // Eq. 1 grows with q when alpha_p >= 0 and T_GEMM does not decrease: then bisect over the candidates.  A profiled table
    // (medians of measurements) or an unconstrained fit need not be monotone; then "the largest that fits" is found the way
    // it is defined, by scanning down from the top.
    bool monotone = model->alpha_p_ms >= 0.0 && std::isfinite(model->alpha_p_ms);
    for (int i = 0; monotone && i < model->n_gemm; ++i)
        monotone = std::isfinite(model->gemm_ms[i]) && (i == 0 || model->gemm_ms[i] >= model->gemm_ms[i - 1]);
    if (!monotone) {
        for (int64_t k = hi; k >= 1; --k)
            if (fits(k * granularity)) {
                *out_q = k * granularity;
                return SA_OK;
            }
        return SA_OK;
    }
    while (lo < hi) {
        const int64_t mid = (lo + hi + 1) / 2;
        if (fits(mid * granularity)) lo = mid; else hi = mid - 1;
    }
    *out_q = lo * granularity;
    return SA_OK;
}

extern "C" int32_t sa_latency_fit(const float *ms, const int64_t *sum_kv, int32_t n, int32_t with_intercept,
                                  sa_latency_model *out, double *out_max_rel_err) {
    if (!ms || !sum_kv || !out || n <= 0) return SA_ERR_INVALID_ARG;
    // columns: [1] sum_L sum_A, each scaled by its largest magnitude; all-zero columns carry no information
    double scale[3] = {1.0, 0.0, 0.0};
    for (int32_t i = 0; i < n; ++i) {
        scale[1] = fmax(scale[1], fabs(double(sum_kv[2 * i])));
        scale[2] = fmax(scale[2], fabs(double(sum_kv[2 * i + 1])));
    }
    int cols[3], nc = 0;
    if (with_intercept) cols[nc++] = 0;
    if (scale[1] > 0) cols[nc++] = 1;
    if (scale[2] > 0) cols[nc++] = 2;
    double coef[3] = {0.0, 0.0, 0.0};
    if (nc > 0) {
        double a[3][4] = {};
        for (int32_t i = 0; i < n; ++i) {
            const double row[3] = {1.0, double(sum_kv[2 * i]) / (scale[1] > 0 ? scale[1] : 1.0),
                                   double(sum_kv[2 * i + 1]) / (scale[2] > 0 ? scale[2] : 1.0)};
            for (int r = 0; r < nc; ++r) {
                for (int c = 0; c < nc; ++c) a[r][c] += row[cols[r]] * row[cols[c]];
                a[r][nc] += row[cols[r]] * double(ms[i]);
            }
        }
        double x[3] = {0.0, 0.0, 0.0};
        if (!solve(nc, a, x)) return SA_ERR_INVALID_ARG;  // collinear profile: not enough distinct points
        for (int r = 0; r < nc; ++r) coef[cols[r]] = x[r] / scale[cols[r]];
    }
    *out = sa_latency_model{};
    out->c0_ms = coef[0];
    out->alpha_d_ms = coef[1];
    out->alpha_p_ms = coef[2];
    out->n_gemm = 0;  // no GEMMs on this path: T_GEMM = 0 until a table is supplied by the caller
    if (out_max_rel_err) {
        double worst = 0.0;
        for (int32_t i = 0; i < n; ++i) {
            const double pred = coef[0] + coef[1] * double(sum_kv[2 * i]) + coef[2] * double(sum_kv[2 * i + 1]);
            const double y = double(ms[i]);
            worst = fmax(worst, fabs(pred - y) / fmax(fabs(y), 1e-300));
        }
        *out_max_rel_err = worst;
    }
    return SA_OK;
}

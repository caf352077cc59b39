// KAIROS' step-latency model (Eq. 4), TBT-safe greedy chunk schedule (Eq. 5-6) and deflection
// decision (Eq. 1-3, 7; Algorithm 1) -- include/kairos.h has the contract and the readings.  Host-only, allocation-free on
// the decision path (the paper measures < 1 ms per decision on one core).
#include <cmath>
#include <cstdint>
#include <limits>

#include "kairos_internal.h"

namespace kairos {
namespace {

inline double eval_t0(const kairos_step_model& m, double B, double Kd) { return m.a[0] + m.a[1] * B + m.a[2] * Kd; }
inline double eval_dt(const kairos_step_model& m, double C, double P, double Kd) {
    if (C <= 0) return 0.0;
    return m.b[0] + m.b[1] * C + m.b[2] * C * (P + 0.5 * (C + 1.0)) + m.b[3] * Kd;
}
inline double eval_step(const kairos_step_model& m, double B, double Kd, double C, double P) {
    return eval_t0(m, B, Kd) + eval_dt(m, C, P, Kd);
}
inline double eval_prefill(const kairos_prefill_model& p, double tokens, double cached) {
    return p.p[0] + p.p[1] * tokens + p.p[2] * cached + p.p[3] * tokens * cached;
}

// Solves the N x N normal equations A x = y in place (Gaussian elimination, partial pivoting).  false = singular.
template <int N>
bool solve(double (&A)[N][N], double (&y)[N]) {
    for (int c = 0; c < N; ++c) {
        int piv = c;
        for (int r = c + 1; r < N; ++r)
            if (std::fabs(A[r][c]) > std::fabs(A[piv][c])) piv = r;
        if (std::fabs(A[piv][c]) < 1e-12) return false;
        if (piv != c) {
            for (int k = 0; k < N; ++k) std::swap(A[piv][k], A[c][k]);
            std::swap(y[piv], y[c]);
        }
        for (int r = c + 1; r < N; ++r) {
            const double f = A[r][c] / A[c][c];
            for (int k = c; k < N; ++k) A[r][k] -= f * A[c][k];
            y[r] -= f * y[c];
        }
    }
    for (int c = N - 1; c >= 0; --c) {
        double s = y[c];
        for (int k = c + 1; k < N; ++k) s -= A[c][k] * y[k];
        y[c] = s / A[c][c];
    }
    return true;
}

// Weighted least squares over rows (phi, target, weight): accumulates the normal equations with every feature divided by
// its largest magnitude (the raw columns span ten orders of magnitude), solves, and scales the coefficients back.
template <int N, class RowFn>
bool weighted_lsq(int32_t n, RowFn row, double (&coef)[N]) {
    double scale[N];
    for (int k = 0; k < N; ++k) scale[k] = 0.0;
    int used = 0;
    for (int32_t i = 0; i < n; ++i) {
        double phi[N], t, w;
        if (!row(i, phi, &t, &w)) continue;
        ++used;
        for (int k = 0; k < N; ++k) scale[k] = std::fmax(scale[k], std::fabs(phi[k]));
    }
    if (used < N) return false;
    for (int k = 0; k < N; ++k)
        if (scale[k] == 0.0) return false;
    double A[N][N], y[N];
    for (int r = 0; r < N; ++r) {
        y[r] = 0.0;
        for (int c = 0; c < N; ++c) A[r][c] = 0.0;
    }
    for (int32_t i = 0; i < n; ++i) {
        double phi[N], t, w;
        if (!row(i, phi, &t, &w)) continue;
        for (int k = 0; k < N; ++k) phi[k] = phi[k] / scale[k] * w;
        t *= w;
        for (int r = 0; r < N; ++r) {
            y[r] += phi[r] * t;
            for (int c = 0; c < N; ++c) A[r][c] += phi[r] * phi[c];
        }
    }
    if (!solve<N>(A, y)) return false;
    for (int k = 0; k < N; ++k) coef[k] = y[k] / scale[k];
    return true;
}

}  // namespace
}  // namespace kairos

using namespace kairos;

extern "C" {

int kairos_fit_latency_model(const int64_t* B, const int64_t* Kd, const int64_t* C, const int64_t* P, const double* T,
                             int32_t n, kairos_step_model* model, double* mape_out) {
    if (!B || !Kd || !C || !P || !T || !model || n < 1) return fail(KAIROS_ERR_INVALID_ARG, "fit: NULL argument or n < 1");
    for (int32_t i = 0; i < n; ++i)
        if (!(T[i] > 0.0) || !std::isfinite(T[i]) || B[i] < 0 || Kd[i] < 0 || C[i] < 0 || P[i] < 0)
            return fail(KAIROS_ERR_INVALID_ARG, "fit: sample " + std::to_string(i) + " has T <= 0 or a negative coordinate");
    kairos_step_model m{};
    // T0 from the decode-only samples
    auto row0 = [&](int32_t i, double* phi, double* t, double* w) {
        if (C[i] != 0) return false;
        phi[0] = 1.0; phi[1] = double(B[i]); phi[2] = double(Kd[i]);
        *t = T[i]; *w = 1.0 / T[i];
        return true;
    };
    if (!weighted_lsq<3>(n, row0, m.a)) return fail(KAIROS_ERR_INVALID_ARG, "fit: decode-only samples do not determine T0 (need >= 3, varying B and Kd)");
    // dT_pf from the residual of the mixed samples
    auto row1 = [&](int32_t i, double* phi, double* t, double* w) {
        if (C[i] == 0) return false;
        const double c = double(C[i]);
        phi[0] = 1.0; phi[1] = c; phi[2] = c * (double(P[i]) + 0.5 * (c + 1.0)); phi[3] = double(Kd[i]);
        *t = T[i] - eval_t0(m, double(B[i]), double(Kd[i]));
        *w = 1.0 / T[i];
        return true;
    };
    if (!weighted_lsq<4>(n, row1, m.b)) return fail(KAIROS_ERR_INVALID_ARG, "fit: mixed samples do not determine dT_pf (need >= 4, varying C, P and Kd)");
    *model = m;
    if (mape_out) {
        double s = 0.0;
        for (int32_t i = 0; i < n; ++i) s += std::fabs(eval_step(m, double(B[i]), double(Kd[i]), double(C[i]), double(P[i])) - T[i]) / T[i];
        *mape_out = s / n;
    }
    return KAIROS_OK;
}

double kairos_predict_step(const kairos_step_model* model, int64_t B, int64_t Kd, int64_t C, int64_t P) {
    if (!model) return std::numeric_limits<double>::quiet_NaN();
    return eval_step(*model, double(B), double(Kd), double(C), double(P));
}

int kairos_decide(const kairos_step_model* model, const kairos_prefill_model* prefill, const kairos_decide_input* in,
                  int32_t* schedule_out, int32_t max_schedule, kairos_decide_output* out) {
    if (!model || !prefill || !in || !out) return fail(KAIROS_ERR_INVALID_ARG, "decide: NULL argument");
    if (in->prompt_len < 1 || in->chi_p < 1 || in->n_queue < 0 || in->n_nodes < 0 || in->n_candidates < 1 || max_schedule < 0)
        return fail(KAIROS_ERR_INVALID_ARG, "decide: bad size");
    if ((in->n_queue > 0 && !in->queue_lens) || (in->n_nodes > 0 && (!in->node_B || !in->node_K)) || !in->candidates)
        return fail(KAIROS_ERR_INVALID_ARG, "decide: NULL array");
    if (!(in->beta > 0.0) || !(in->alpha >= 1.0)) return fail(KAIROS_ERR_INVALID_ARG, "decide: beta must be > 0 and alpha >= 1");
    for (int32_t c = 0; c < in->n_candidates; ++c)
        if (in->candidates[c] < 1 || (c > 0 && in->candidates[c] >= in->candidates[c - 1]))
            return fail(KAIROS_ERR_INVALID_ARG, "decide: candidates must be positive and strictly decreasing");
    for (int32_t n = 0; n < in->n_nodes; ++n)
        if (in->node_B[n] < 0 || in->node_K[n] < 0) return fail(KAIROS_ERR_INVALID_ARG, "decide: negative node state");

    // 1. prefill-node TTFT estimate, Eq. 1-3
    double queued = 0.0;
    for (int32_t i = 0; i < in->n_queue; ++i) queued += double(in->queue_lens[i]);
    const double w_queue = queued / in->chi_p * eval_prefill(*prefill, in->chi_p, queued / 2.0);            // Eq. 2
    double t_pf = 0.0;
    const int32_t n_pf_steps = (in->prompt_len + in->chi_p - 1) / in->chi_p;
    for (int32_t i = 0; i < n_pf_steps; ++i) t_pf += eval_prefill(*prefill, in->chi_p, double(in->chi_p) * i);  // Eq. 3 (G19)
    const double est_pf = w_queue + t_pf;                                                                  // Eq. 1

    // 2. a TBT-safe schedule per decode node; 3. the fastest feasible one.  The schedule of a node is a deterministic
    // function of its state, so the best node's schedule is rebuilt into schedule_out at the end instead of being stored.
    const double limit = in->beta * in->tbt_slo;
    auto walk = [&](int32_t n, int32_t* sched, int32_t cap, int32_t* steps_out, double* ttft_out) {
        const double B = double(in->node_B[n]);
        double Kd = double(in->node_K[n]);
        int64_t served = 0;
        int32_t steps = 0;
        double ttft = 0.0;
        while (served < in->prompt_len) {
            int32_t chi = 0;
            double t = 0.0;
            for (int32_t c = 0; c < in->n_candidates; ++c) {  // LargestSafe: first chi in X (decreasing) satisfying Eq. 5
                const int32_t cand = in->candidates[c];
                if (cand <= in->node_B[n]) break;             // carries no prefill token; so does every smaller one
                t = eval_step(*model, B, Kd, double(cand) - B, double(served));
                if (t <= limit) { chi = cand; break; }
            }
            if (chi == 0) return false;                       // node n infeasible
            if (sched && steps < cap) sched[steps] = chi;
            ++steps;
            ttft += t;                                        // Eq. 6
            Kd += B;
            served += chi - in->node_B[n];
        }
        *steps_out = steps;
        *ttft_out = ttft;
        return true;
    };
    int32_t best_n = -1, best_steps = 0;
    double best_ttft = std::numeric_limits<double>::infinity();
    for (int32_t n = 0; n < in->n_nodes; ++n) {
        int32_t steps;
        double ttft;
        if (walk(n, nullptr, 0, &steps, &ttft) && ttft < best_ttft) { best_ttft = ttft; best_n = n; best_steps = steps; }
    }
    out->ttft_pf = est_pf;
    out->ttft_dec = best_ttft;
    out->decision = 0;
    out->node = -1;
    out->n_steps = 0;
    // 4. deflect only if the margin holds, Eq. 7
    if (best_n >= 0 && best_ttft <= in->alpha * est_pf && best_ttft <= in->ttft_slo) {
        out->n_steps = best_steps;
        if (schedule_out && best_steps > max_schedule)
            return fail(KAIROS_ERR_WORKSPACE, "decide: schedule has " + std::to_string(best_steps) + " steps, schedule_out holds fewer");
        int32_t steps;
        double ttft;
        if (schedule_out) walk(best_n, schedule_out, max_schedule, &steps, &ttft);
        out->decision = 1;
        out->node = best_n;
    }
    return KAIROS_OK;
}

}  // extern "C"

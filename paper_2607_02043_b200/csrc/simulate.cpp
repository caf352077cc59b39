// SURVEY.md 8(f) row 4 (second half): the paper's policy simulator (section 3.4) -- the
// latency models of Eq. 3-4 wrapped in an event loop over N_p FIFO prefill nodes and N_d decode nodes, with the static
// deflection policies SQ(theta) / SL(l), the no-deflection baseline and the Oracle (Algorithm 1 on the simulator's own
// state).  Host-only.  The paper gives no pseudo-code; include/kairos.h states the event rules (reading G22).
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <limits>
#include <vector>

#include "kairos_internal.h"

namespace {

struct Active { int32_t req; int64_t context; int32_t remaining; };
struct Pending { int32_t req; double ready; };
struct Deflected { int32_t req = -1; int64_t served = 0; std::vector<int32_t> sched; int32_t step = 0; int32_t cur = 0; bool has_sched = false; };

inline double t0_of(const kairos_step_model& m, double B, double Kd) { return m.a[0] + m.a[1] * B + m.a[2] * Kd; }
inline double dt_of(const kairos_step_model& m, double C, double P, double Kd) {
    if (C <= 0) return 0.0;
    return m.b[0] + m.b[1] * C + m.b[2] * C * (P + 0.5 * (C + 1.0)) + m.b[3] * Kd;
}
inline double pf_step(const kairos_prefill_model& p, double tokens, double cached) {
    return p.p[0] + p.p[1] * tokens + p.p[2] * cached + p.p[3] * tokens * cached;
}

}  // namespace

extern "C" int kairos_simulate(const kairos_step_model* model, const kairos_prefill_model* prefill, const kairos_sim_config* cfg,
                               const kairos_sim_request* reqs, int32_t n, double* ttft_out, kairos_sim_result* out) {
    using kairos::fail;
    if (!model || !prefill || !cfg || !out || (n > 0 && !reqs) || n < 0) return fail(KAIROS_ERR_INVALID_ARG, "simulate: NULL argument or n < 0");
    if (cfg->n_prefill < 1 || cfg->n_decode < 1 || cfg->chi_p < 1 || cfg->policy < 0 || cfg->policy > 3 || cfg->static_chi < 1)
        return fail(KAIROS_ERR_INVALID_ARG, "simulate: bad configuration");
    if (cfg->policy == 3 && (!cfg->candidates || cfg->n_candidates < 1)) return fail(KAIROS_ERR_INVALID_ARG, "simulate: the Oracle policy needs candidates");
    for (int32_t r = 0; r < n; ++r)
        if (reqs[r].prompt_len < 1 || reqs[r].output_len < 0 || (r > 0 && reqs[r].arrival < reqs[r - 1].arrival) || !(reqs[r].arrival >= 0.0))
            return fail(KAIROS_ERR_INVALID_ARG, "simulate: requests must have prompt_len >= 1, output_len >= 0 and be sorted by arrival");
    const double inf = std::numeric_limits<double>::infinity();
    const int32_t NP = cfg->n_prefill, ND = cfg->n_decode;
    std::vector<std::vector<int32_t>> pf_queue(NP);
    std::vector<int32_t> pf_cur(NP, -1);
    std::vector<double> pf_end(NP, inf);
    std::vector<std::vector<Active>> active(ND);
    std::vector<std::vector<Pending>> pending(ND);
    std::vector<Deflected> defl(ND);
    std::vector<double> step_end(ND, inf);
    std::vector<double> ttft(size_t(n), inf);
    std::vector<char> violated(size_t(n), 0);
    int32_t n_deflected = 0, finished = 0, next_arr = 0;
    int64_t decode_steps = 0, violations = 0;
    double t = 0.0;
    std::vector<int32_t> qlens, node_B, elig, sched(4096);
    std::vector<int64_t> node_K;

    auto t_pf = [&](int32_t l) {
        double s = 0.0;
        const int32_t steps = (l + cfg->chi_p - 1) / cfg->chi_p;
        for (int32_t i = 0; i < steps; ++i) s += pf_step(*prefill, cfg->chi_p, double(cfg->chi_p) * i);
        return s;
    };
    auto outstanding = [&](int32_t i) {
        int64_t s = 0;
        for (int32_t r : pf_queue[i]) s += reqs[r].prompt_len;
        return s + (pf_cur[i] >= 0 ? reqs[pf_cur[i]].prompt_len : 0);
    };

    while (finished < n) {
        // ---- next event time
        double t_next = next_arr < n ? reqs[next_arr].arrival : inf;
        for (int32_t i = 0; i < NP; ++i) t_next = std::min(t_next, pf_end[i]);
        for (int32_t d = 0; d < ND; ++d) t_next = std::min(t_next, step_end[d]);
        for (int32_t d = 0; d < ND; ++d)
            if (step_end[d] == inf && !pending[d].empty()) {
                double first = inf;
                for (const Pending& q : pending[d]) first = std::min(first, q.ready);
                t_next = std::min(t_next, std::max(t, first));
            }
        if (!(t_next < inf)) return fail(KAIROS_ERR_INVALID_ARG, "simulate: stalled (no event left but requests unfinished)");
        t = t_next;
        // ---- decode step ends
        for (int32_t d = 0; d < ND; ++d) {
            if (step_end[d] != t) continue;
            step_end[d] = inf;
            size_t k = 0;
            for (Active& e : active[d]) {
                e.context += 1;
                e.remaining -= 1;
                if (e.remaining > 0) active[d][k++] = e;
                else ++finished;
            }
            active[d].resize(k);
            if (defl[d].req >= 0) {
                const int32_t r = defl[d].req;
                defl[d].served += defl[d].cur;
                defl[d].step += 1;
                if (defl[d].served >= reqs[r].prompt_len) {
                    ttft[r] = t - reqs[r].arrival;
                    pending[d].push_back(Pending{r, t});
                    defl[d] = Deflected();
                }
            }
        }
        // ---- prefill completions
        for (int32_t i = 0; i < NP; ++i) {
            if (pf_end[i] != t) continue;
            const int32_t r = pf_cur[i];
            pf_cur[i] = -1;
            pf_end[i] = inf;
            const double ready = t + cfg->transfer_per_token * reqs[r].prompt_len;
            ttft[r] = ready - reqs[r].arrival;
            int32_t best = 0;
            size_t best_load = active[0].size() + pending[0].size();
            for (int32_t d = 1; d < ND; ++d) {
                const size_t load = active[d].size() + pending[d].size();
                if (load < best_load) { best_load = load; best = d; }
            }
            pending[best].push_back(Pending{r, ready});
        }
        // ---- the arrival(s) at this instant
        while (next_arr < n && reqs[next_arr].arrival == t) {
            const int32_t r = next_arr++;
            const int32_t l = reqs[r].prompt_len;
            int32_t pn = 0;
            int64_t pn_out = outstanding(0);
            for (int32_t i = 1; i < NP; ++i) {
                const int64_t o = outstanding(i);
                if (o < pn_out) { pn_out = o; pn = i; }
            }
            elig.clear();
            for (int32_t d = 0; d < ND; ++d)
                if (defl[d].req < 0) elig.push_back(d);
            auto least_loaded = [&]() {
                int32_t best = elig[0];
                for (int32_t d : elig)
                    if (active[d].size() < active[best].size()) best = d;
                return best;
            };
            int32_t target = -1, sched_len = 0;
            if (cfg->policy == 1) {
                bool all = true;
                for (int32_t i = 0; i < NP; ++i) all = all && int64_t(pf_queue[i].size()) > int64_t(cfg->param);
                if (all && !elig.empty()) target = least_loaded();
            } else if (cfg->policy == 2) {
                if (l < cfg->param && !elig.empty()) target = least_loaded();
            } else if (cfg->policy == 3 && !elig.empty()) {
                qlens.clear();
                if (pf_cur[pn] >= 0) qlens.push_back(reqs[pf_cur[pn]].prompt_len);
                for (int32_t q : pf_queue[pn]) qlens.push_back(reqs[q].prompt_len);
                node_B.clear();
                node_K.clear();
                for (int32_t d : elig) {
                    int64_t kd = 0;
                    for (const Active& e : active[d]) kd += e.context;
                    node_B.push_back(int32_t(active[d].size()));
                    node_K.push_back(kd);
                }
                kairos_decide_input in{};
                in.prompt_len = l;
                in.queue_lens = qlens.data();
                in.n_queue = int32_t(qlens.size());
                in.chi_p = cfg->chi_p;
                in.node_B = node_B.data();
                in.node_K = node_K.data();
                in.n_nodes = int32_t(elig.size());
                in.candidates = cfg->candidates;
                in.n_candidates = cfg->n_candidates;
                in.tbt_slo = cfg->tbt_slo;
                in.beta = cfg->beta;
                in.alpha = cfg->alpha;
                in.ttft_slo = cfg->ttft_slo;
                kairos_decide_output dout{};
                int rc = kairos_decide(model, prefill, &in, sched.data(), int32_t(sched.size()), &dout);
                if (rc == KAIROS_ERR_WORKSPACE) {  // a very long schedule: grow and repeat
                    sched.resize(size_t(dout.n_steps));
                    rc = kairos_decide(model, prefill, &in, sched.data(), int32_t(sched.size()), &dout);
                }
                if (rc != KAIROS_OK) return rc;
                if (dout.decision == 1) {
                    target = elig[size_t(dout.node)];
                    sched_len = dout.n_steps;
                }
            }
            if (target >= 0) {
                ++n_deflected;
                Deflected x;
                x.req = r;
                x.has_sched = sched_len > 0;
                if (x.has_sched) x.sched.assign(sched.begin(), sched.begin() + sched_len);
                defl[target] = x;
            } else {
                pf_queue[pn].push_back(r);
            }
        }
        // ---- idle nodes start work
        for (int32_t i = 0; i < NP; ++i)
            if (pf_cur[i] < 0 && !pf_queue[i].empty()) {
                pf_cur[i] = pf_queue[i].front();
                pf_queue[i].erase(pf_queue[i].begin());
                pf_end[i] = t + t_pf(reqs[pf_cur[i]].prompt_len);
            }
        for (int32_t d = 0; d < ND; ++d) {
            if (step_end[d] != inf) continue;
            size_t k = 0;
            for (const Pending& q : pending[d]) {
                if (q.ready <= t) {
                    if (reqs[q.req].output_len > 0) active[d].push_back(Active{q.req, reqs[q.req].prompt_len, reqs[q.req].output_len});
                    else ++finished;
                } else {
                    pending[d][k++] = q;
                }
            }
            pending[d].resize(k);
            const int32_t B = int32_t(active[d].size());
            int32_t C = 0;
            int64_t P = 0;
            if (defl[d].req >= 0) {
                Deflected& x = defl[d];
                P = x.served;
                const int32_t chi = x.has_sched ? x.sched[size_t(std::min<int32_t>(x.step, int32_t(x.sched.size()) - 1))] : cfg->static_chi;
                C = int32_t(std::min<int64_t>(std::max(chi - B, 1), reqs[x.req].prompt_len - P));
                x.cur = C;
            }
            if (B == 0 && C == 0) continue;
            int64_t kd = 0;
            for (const Active& e : active[d]) kd += e.context;
            const double T = t0_of(*model, double(B), double(kd)) + dt_of(*model, double(C), double(P), double(kd));
            step_end[d] = t + T;
            if (B > 0) {
                ++decode_steps;
                if (T > cfg->tbt_slo) {
                    ++violations;
                    for (const Active& e : active[d]) violated[size_t(e.req)] = 1;
                }
            }
        }
    }
    std::vector<double> s(ttft);
    std::sort(s.begin(), s.end());
    int32_t ok = 0;
    double sum = 0.0;
    for (int32_t r = 0; r < n; ++r) {
        sum += ttft[size_t(r)];
        if (ttft[size_t(r)] <= cfg->ttft_slo && !violated[size_t(r)]) ++ok;
    }
    out->n_requests = n;
    out->n_deflected = n_deflected;
    out->p95_ttft = n ? s[size_t(std::max<int64_t>(0, int64_t(std::ceil(0.95 * n)) - 1))] : 0.0;
    out->mean_ttft = n ? sum / n : 0.0;
    out->decode_steps = decode_steps;
    out->tbt_violations = violations;
    out->slo_attainment = n ? double(ok) / n : 1.0;
    out->makespan = t;
    if (ttft_out)
        for (int32_t r = 0; r < n; ++r) ttft_out[r] = ttft[size_t(r)];
    return KAIROS_OK;
}

// cc_control.cu -- host-only: the paper's cost / speed-up model and one decision of its unified layer-wise
// scaling loop.  PAPER.md:151-217 (section 4.2, Eq. 1-10), PAPER.md:290-353 (section
// 4.4, Algorithm 2), PAPER.md:219-288 (section 4.3, Algorithm 1).  No GPU work: the hot path takes `replica_assign` and the replica counts from its caller;
// this is the piece that would choose them.  Readings of what the paper leaves open: DESIGN.md section 7c.
#include "../../include/cocoscale.h"

#include <algorithm>
#include <cmath>
#include <vector>

extern "C" {

// Eq. 1: C_mem(N, P) ~ N * kappa * (12 d^2 + bs / P * l * d)
double cc_ctl_mem_bytes(int N, int P, int bs, int l, int d_hidden, double kappa) {
    const double d = d_hidden;
    return (double)N * kappa * (12.0 * d * d + (double)bs / P * l * d);
}

// Eq. 2: C_comp(N, P) ~ N / P * 24 * bs * l * d^2
double cc_ctl_flops(int N, int P, int bs, int l, int d_hidden) {
    const double d = d_hidden;
    return (double)N / P * 24.0 * bs * l * d * d;
}

// Eq. 5 with the bytes-per-element factor the paper omits (reading G2): T(P) ~ 2 * (bs / P * (P - 1) * l * d * kappa) / B
double cc_ctl_comm_seconds(int P, int bs, int l, int d_hidden, double kappa, double bandwidth_bytes_per_s) {
    return 2.0 * ((double)bs / P * (P - 1) * l * d_hidden * kappa) / bandwidth_bytes_per_s;
}

// Eq. 7: S(N, P) = 1 / (1 - alpha + alpha / P + beta), alpha = N / L, beta = T(P) / (L * t_comp)
double cc_ctl_speedup(int L, int N, int P, double beta) {
    const double alpha = (double)N / L;
    return 1.0 / (1.0 - alpha + alpha / P + beta);
}

// Eq. 8-10, homogeneous devices: W(v) = sum_l t_comp * ceil(bs / v_l) / bs; T(v) = sum over the indices where v
// changes (the boundaries of the model count as v = 1) of 2 * ceil(bs * (v - 1) / v) * d * kappa / B with v the
// larger degree at that boundary; S(v) = L * t_comp / (W + T).
double cc_ctl_speedup_vec(const int32_t* v, int L, int bs, double t_comp_s, int d_hidden, double kappa,
                          double bandwidth_bytes_per_s) {
    double W = 0.0, T = 0.0;
    for (int l = 0; l < L; ++l) W += t_comp_s * (double)((bs + v[l] - 1) / v[l]) / bs;
    for (int l = 0; l <= L; ++l) {
        const int a = l == 0 ? 1 : v[l - 1], b = l == L ? 1 : v[l];
        if (a == b) continue;
        const int hi = std::max(a, b);
        T += 2.0 * std::ceil((double)bs * (hi - 1) / hi) * d_hidden * kappa / bandwidth_bytes_per_s;
    }
    return (double)L * t_comp_s / (W + T);
}

// Dist of Algorithm 2 for configurations given as (N, P): L1 distance of the vectors v (N entries equal to P, the
// rest 1) when the shorter replicated segment is nested in the longer one.
int cc_ctl_distance(int N0, int P0, int N1, int P1) {
    const int common = std::min(N0, N1);
    return common * std::abs(P1 - P0) + std::max(0, N1 - N0) * (P1 - 1) + std::max(0, N0 - N1) * (P0 - 1);
}

int cc_ctl_candidate_count(int L, int P_max) { return L * P_max; }

// One pass of Algorithm 2's body for one instance (lines 3-19).
cc_status cc_ctl_decide(const cc_ctl_params* p, int N_cur, int P_cur, double latency, double* cold_capacity, int* N_new,
                        int* P_new, cc_ctl_action* action) {
    if (!p || !cold_capacity || !N_new || !P_new || !action || p->L < 1 || p->P_max < 1 || p->P_max > CC_MAX_REPLICAS ||
        !(p->slo > 0.0) || N_cur < 0 || N_cur > p->L || P_cur < 1 || P_cur > p->P_max)
        return CC_ERR_INVALID;
    *N_new = N_cur;
    *P_new = P_cur;
    *action = CC_CTL_NONE;
    if (std::fabs(latency - p->slo) / p->slo <= p->delta) return CC_OK;                      // line 3
    auto S = [&](int N, int P) { return cc_ctl_speedup(p->L, N, P, p->beta[P]); };
    auto cost = [&](int N, int P) { return p->cost_per_device * (P - 1) + p->cost_per_layer_copy * N * (P - 1); };
    const double alpha_req = S(N_cur, P_cur) * (latency / p->slo);                            // lines 4-5
    struct Cand { int dist, N, P; };
    std::vector<Cand> cand;
    for (int N = 1; N <= p->L; ++N)
        for (int P = 1; P <= p->P_max; ++P)
            if (S(N, P) >= alpha_req) cand.push_back({cc_ctl_distance(N_cur, P_cur, N, P), N, P});   // line 6
    std::sort(cand.begin(), cand.end(), [](const Cand& a, const Cand& b) {                    // line 7 (ties: N, then P)
        return a.dist != b.dist ? a.dist < b.dist : (a.N != b.N ? a.N < b.N : a.P < b.P);
    });
    for (const Cand& c : cand) {                                                              // lines 9-16
        const double d_res = cost(c.N, c.P) - cost(N_cur, P_cur);
        if (d_res <= 0.0 || *cold_capacity >= d_res) {
            *cold_capacity -= d_res;
            *N_new = c.N;
            *P_new = c.P;
            *action = CC_CTL_UPDATED;
            return CC_OK;
        }
    }
    if (latency > p->slo) *action = CC_CTL_INSTANCE_SCALE;                                    // lines 17-19
    return CC_OK;
}

// Algorithm 1: initial global placement, a priority-greedy pass over the instances.
// Line 3: the pool is the devices with Load < tau_idle.  Lines 4-7: instances by descending Priority = load -
// capacity (Eq. 11; ties: lower index first).  Lines 10-17: every (N, P), 1 <= N <= L, 2 <= P <= P_max, whose
// per-device memory C_mem(N, P) (Eq. 1) fits on at least P - 1 pool devices is feasible.  Line 19: the feasible
// candidate of largest S(N, P) wins (ties: fewer devices, then fewer layers); its devices are the P - 1 of largest
// free memory among those that fit (ties: lower index) and leave the pool (line 21).
cc_status cc_ctl_place(const cc_ctl_params* p, const cc_ctl_instance* inst, int n_inst, const cc_ctl_device* dev, int n_dev,
                       double tau_idle, cc_ctl_placement* out, int* n_out) {
    if (!p || !inst || !dev || !out || !n_out || n_inst < 0 || n_dev < 0 || p->P_max < 1 || p->P_max > CC_MAX_REPLICAS)
        return CC_ERR_INVALID;
    for (int k = 0; k < n_inst; ++k)
        if (inst[k].L < 1 || inst[k].bs < 1 || inst[k].l < 0 || inst[k].d_hidden < 1 || !(inst[k].kappa > 0.0)) return CC_ERR_INVALID;
    std::vector<char> in_pool((size_t)n_dev);
    for (int d = 0; d < n_dev; ++d) in_pool[d] = dev[d].load < tau_idle;                      // line 3
    std::vector<int> order((size_t)n_inst);
    for (int k = 0; k < n_inst; ++k) order[k] = k;
    std::stable_sort(order.begin(), order.end(), [&](int a, int b) {                          // lines 4-7
        return inst[a].load - inst[a].capacity > inst[b].load - inst[b].capacity;
    });
    int n = 0;
    for (int k : order) {                                                                     // line 9
        const cc_ctl_instance& I = inst[k];
        double best_s = 0.0;
        int best_N = 0, best_P = 0;
        for (int N = 1; N <= I.L; ++N)
            for (int P = 2; P <= p->P_max; ++P) {                                             // line 10
                const double need = cc_ctl_mem_bytes(N, P, I.bs, I.l, I.d_hidden, I.kappa);  // line 11
                int fit = 0;
                for (int d = 0; d < n_dev; ++d) fit += in_pool[d] && dev[d].free_mem_bytes >= need;   // line 12
                if (fit < P - 1) continue;                                                    // line 13
                const double s = cc_ctl_speedup(I.L, N, P, p->beta[P]);
                // speed-ups that agree to 1e-12 are a tie (N (1 - 1/P) takes the same value for many pairs when beta = 0)
                const bool tie = best_P != 0 && std::fabs(s - best_s) <= 1e-12 * best_s;
                if (best_P == 0 || (!tie && s > best_s) || (tie && (P < best_P || (P == best_P && N < best_N)))) {
                    best_s = s; best_N = N; best_P = P;                                       // line 19
                }
            }
        if (best_P == 0) continue;                                                            // line 18
        const double need = cc_ctl_mem_bytes(best_N, best_P, I.bs, I.l, I.d_hidden, I.kappa);
        cc_ctl_placement& pl = out[n++];
        pl.instance = k; pl.N = best_N; pl.P = best_P; pl.speedup = best_s;
        for (int j = 0; j < CC_MAX_REPLICAS - 1; ++j) pl.devices[j] = -1;
        for (int j = 0; j < best_P - 1; ++j) {                                                // line 14, largest idle memory first
            int pick = -1;
            for (int d = 0; d < n_dev; ++d)
                if (in_pool[d] && dev[d].free_mem_bytes >= need && (pick < 0 || dev[d].free_mem_bytes > dev[pick].free_mem_bytes)) pick = d;
            pl.devices[j] = pick;
            in_pool[pick] = 0;                                                                // line 21
        }
    }
    *n_out = n;
    return CC_OK;
}

}  // extern "C"

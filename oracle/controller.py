"""oracle/controller.py -- TEST INFRASTRUCTURE: the paper's cost / speed-up model (Eq. 1-10) and
one pass of Algorithm 2 written out plainly, independently of the library's cc_control.cu:
distances are taken on explicit configuration vectors v, candidates are a sorted list of tuples.
Readings: the replicated segment of the shorter configuration is nested in the longer one;
ties in the distance are broken by smaller N, then smaller P; Cost(N, P) = c_dev*(P-1) + c_copy*N*(P-1);
Eq. 5 gets the bytes-per-element factor kappa; model boundaries count as v = 1 in Eq. 9."""
from __future__ import annotations

import math


def mem_bytes(N, P, bs, l, d, kappa):                      # Eq. 1
    return N * kappa * (12 * d * d + bs / P * l * d)


def flops(N, P, bs, l, d):                                 # Eq. 2
    return N / P * 24 * bs * l * d * d


def comm_seconds(P, bs, l, d, kappa, B):                   # Eq. 5 (x kappa)
    return 2 * (bs / P * (P - 1) * l * d * kappa) / B


def speedup(L, N, P, beta):                                # Eq. 6 with t_comp = 1, T = beta * L
    return L / ((L - N) + N / P + beta * L)


def vector(L, N, P):
    return [P] * N + [1] * (L - N)


def speedup_vec(v, bs, t_comp, d, kappa, B):               # Eq. 8-10, homogeneous
    L = len(v)
    W = sum(t_comp * math.ceil(bs / x) / bs for x in v)
    ext = [1] + list(v) + [1]
    T = sum(2 * math.ceil(bs * (max(a, b) - 1) / max(a, b)) * d * kappa / B for a, b in zip(ext, ext[1:]) if a != b)
    return L * t_comp / (W + T)


def distance(L, N0, P0, N1, P1):                           # ||v_new - v_cur||_1 on explicit vectors
    return sum(abs(a - b) for a, b in zip(vector(L, N0, P0), vector(L, N1, P1)))


def decide(L, P_max, slo, delta, beta, c_dev, c_copy, N_cur, P_cur, latency, cold):
    """-> (action, N, P, cold) with action in {"none", "updated", "instance_scale"} (Alg. 2 lines 3-19)."""
    if abs(latency - slo) / slo <= delta:
        return "none", N_cur, P_cur, cold
    S = lambda N, P: speedup(L, N, P, beta[P])
    cost = lambda N, P: c_dev * (P - 1) + c_copy * N * (P - 1)
    alpha_req = S(N_cur, P_cur) * (latency / slo)
    cand = sorted((distance(L, N_cur, P_cur, N, P), N, P) for N in range(1, L + 1) for P in range(1, P_max + 1)
                  if S(N, P) >= alpha_req)
    for _, N, P in cand:
        d_res = cost(N, P) - cost(N_cur, P_cur)
        if d_res <= 0 or cold >= d_res:
            return "updated", N, P, cold - d_res
    return ("instance_scale" if latency > slo else "none"), N_cur, P_cur, cold


def place(P_max, beta, instances, devices, tau_idle):
    """Algorithm 1 written as list operations.  instances: dicts with L, bs, l, d, kappa, load,
    capacity; devices: dicts with load, free_mem.  -> [(instance index, N, P, [device indices], S)].
    Readings: equal priorities keep their input order; speed-ups equal to 1e-12 relative are ties, won
    by fewer devices, then fewer layers; the devices are those of largest free memory that fit, lower index first."""
    pool = [i for i, d in enumerate(devices) if d["load"] < tau_idle]                          # line 3
    order = sorted(range(len(instances)), key=lambda k: -(instances[k]["load"] - instances[k]["capacity"]))   # lines 4-7 (stable)
    plan = []
    for k in order:
        I = instances[k]
        feasible = []
        for N in range(1, I["L"] + 1):
            for P in range(2, P_max + 1):
                need = mem_bytes(N, P, I["bs"], I["l"], I["d"], I["kappa"])                  # Eq. 1
                fits = [i for i in pool if devices[i]["free_mem"] >= need]
                if len(fits) >= P - 1:
                    fits.sort(key=lambda i: (-devices[i]["free_mem"], i))
                    feasible.append((speedup(I["L"], N, P, beta[P]), N, P, fits[:P - 1]))
        if not feasible:
            continue
        top = max(f[0] for f in feasible)
        ties = [f for f in feasible if abs(f[0] - top) <= 1e-12 * top]
        s, N, P, devs = min(ties, key=lambda f: (f[2], f[1]))
        plan.append((k, N, P, devs, s))
        pool = [i for i in pool if i not in devs]                                            # line 21
    return plan

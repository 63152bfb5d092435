/*
 * oracle/cc_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT.
 *
 * Plain, slow, obviously-correct CPU statement of what the replicated decoder-layer hot path
 * computes (BASELINE.json north_star).  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may load this.
 * It shares no code, header, table or constant generator with the CUDA library.
 *
 * What the paper fixes (PAPER.md = /root/reference/PAPER.md at survey time):
 *   - a replica is a byte copy of the layer's weights           (PAPER.md:91,  section 3.1)
 *   - the batch is split into sub-batches, each processed by one replica, independently,
 *     and the results are merged (concatenated along batch) in request order
 *
 *   - new K/V entries are appended locally by the replica
 *   - the MLP is SwiGLU
 *   - outputs are bit-wise consistent with the unreplicated run
 * The paper gives NO formula for the layer itself; its composition (pre-norm RMSNorm -> QKV ->
 * RoPE -> paged GQA decode attention -> O-proj + residual -> RMSNorm -> SwiGLU -> down +
 * residual) is BASELINE.json's north_star, with the readings listed in DESIGN.md ("Readings").
 *
 * Precision (north_star: "plain CPU oracle in fp32"): inputs are bf16 widened to fp32, every
 * stored intermediate is fp32, every reduction (dot product, mean of squares, softmax sum) and
 * every transcendental (RoPE angle, cos/sin, exp, rsqrt) is evaluated in fp64 and rounded once
 * to fp32.  bf16 rounding (round-to-nearest-even) happens in exactly two places: the K/V values
 * appended to the cache, and the layer output.
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): naive pure-Python triple loop, identity/one-hot
 * weights, torch-CPU library ops on cfg1, RMSNorm closed forms, RoPE group law / relative-position
 * property / hand value, softmax sum = 1, context-of-1 returns V, equal-K mean, GQA head map,
 * page-reshuffle invariance, SiLU hand values, replicated == unreplicated bitwise.
 * Whole layer: "parity unpinned" by the paper (it prints no activations); pinned only by
 * composition of the above and by an independent torch-CPU restatement on cfg1.
 *
 * No blocking, fusion or reordering: every loop below is the definition written out.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef struct {
    int32_t hidden, n_q_heads, n_kv_heads, head_dim, ffn, page;
    float rms_eps;
    float rope_base;
} orc_desc;

typedef struct { /* bf16 bit patterns, [out][in] row-major */
    const uint16_t *g1, *wq, *wk, *wv, *wo, *g2, *wgate, *wup, *wdown;
} orc_weights;

typedef struct { /* optional fp32 taps, original row order; any pointer may be NULL */
    float *x;      /* [B][d]        a1  input RMSNorm output                    */
    float *q;      /* [B][Hq*Dh]    a3  q after RoPE                            */
    float *k_new;  /* [B][Hkv*Dh]   a3  k after RoPE, before bf16 rounding      */
    float *v_new;  /* [B][Hkv*Dh]   a2  v before bf16 rounding                  */
    float *o;      /* [B][Hq*Dh]    a5  attention output                        */
    float *h1;     /* [B][d]        a6  hidden + O-projection                   */
    float *y;      /* [B][d]        a7  post-attention RMSNorm                  */
    float *a;      /* [B][F]        a8  silu(gate) * up                         */
    float *out;    /* [B][d]        a9  before the final bf16 rounding          */
} orc_taps;

/* ---- bf16 <-> fp32 (bit level) --------------------------------------------------------- */
float orc_bf16_to_f32(uint16_t u) {
    uint32_t w = (uint32_t)u << 16;
    float f;
    memcpy(&f, &w, 4);
    return f;
}

uint16_t orc_f32_to_bf16(float f) { /* round to nearest even */
    uint32_t w;
    memcpy(&w, &f, 4);
    if ((w & 0x7fffffffu) > 0x7f800000u) return (uint16_t)((w >> 16) | 0x40u);
    uint32_t lsb = (w >> 16) & 1u;
    w += 0x7fffu + lsb;
    return (uint16_t)(w >> 16);
}

int orc_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void orc_set_num_threads(int n) {
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

/* ---- a1 / a7: RMSNorm.  x = h * rsqrt(mean(h^2) + eps) * g  (north_star; reading #1) --------- */
void orc_rmsnorm(const float *h, const uint16_t *g, int rows, int d, float eps, float *x) {
    for (int r = 0; r < rows; ++r) {
        double ss = 0.0;
        for (int i = 0; i < d; ++i) ss += (double)h[(size_t)r * d + i] * (double)h[(size_t)r * d + i];
        double inv = 1.0 / sqrt(ss / (double)d + (double)eps);
        for (int i = 0; i < d; ++i)
            x[(size_t)r * d + i] = (float)((double)h[(size_t)r * d + i] * inv * (double)orc_bf16_to_f32(g[i]));
    }
}

/* ---- a2 / a6 / a8 / a9: Y[m][n] = sum_k X[m][k] * W[n][k]   (no bias; reading #3) ------------ */
void orc_matmul_wt(const float *X, const uint16_t *W, int M, int K, int N, float *Y) {
#pragma omp parallel for schedule(static)
    for (int n = 0; n < N; ++n) {
        for (int m = 0; m < M; ++m) {
            double acc = 0.0;
            for (int k = 0; k < K; ++k)
                acc += (double)X[(size_t)m * K + k] * (double)orc_bf16_to_f32(W[(size_t)n * K + k]);
            Y[(size_t)m * N + n] = (float)acc;
        }
    }
}

/* ---- a3: RoPE, rotate-half pairing (i, i + Dh/2), theta_i = base^(-2i/Dh)  (reading #4) ------- */
void orc_rope(float *u, int n_heads, int Dh, int pos, float base) {
    int half = Dh / 2;
    for (int h = 0; h < n_heads; ++h) {
        float *v = u + (size_t)h * Dh;
        for (int i = 0; i < half; ++i) {
            double th = (double)pos * pow((double)base, -2.0 * (double)i / (double)Dh);
            double c = cos(th), s = sin(th);
            double a = (double)v[i], b = (double)v[i + half];
            v[i] = (float)(a * c - b * s);
            v[i + half] = (float)(b * c + a * s);
        }
    }
}

/* ---- a5: paged GQA decode attention for one request  (readings #5-#8, #12, #13) ---------------
 * pools: bf16 [n_pages][Hkv][page][Dh]; bt_row: int32 page ids for this request (pad -1, never
 * dereferenced for t < s); s = tokens attended.  w_out (optional) receives the softmax weights
 * [Hq][s].  kv head of query head hq is hq / G, G = Hq / Hkv. */
int orc_attention_decode(const float *q, const uint16_t *k_pool, const uint16_t *v_pool,
                         const int32_t *bt_row, int s, int Hq, int Hkv, int Dh, int page,
                         float *o, float *w_out) {
    int G = Hq / Hkv;
    double *sc = (double *)malloc(sizeof(double) * (size_t)(s > 0 ? s : 1));
    if (!sc) return -1;
    for (int hq = 0; hq < Hq; ++hq) {
        int hk = hq / G;
        const float *qh = q + (size_t)hq * Dh;
        double mx = -INFINITY;
        for (int t = 0; t < s; ++t) {
            int32_t pg = bt_row[t / page];
            if (pg < 0) { free(sc); return -2; }
            const uint16_t *kr = k_pool + (((size_t)pg * Hkv + hk) * page + (size_t)(t % page)) * Dh;
            double acc = 0.0;
            for (int i = 0; i < Dh; ++i) acc += (double)qh[i] * (double)orc_bf16_to_f32(kr[i]);
            sc[t] = acc / sqrt((double)Dh);
            if (sc[t] > mx) mx = sc[t];
        }
        double sum = 0.0;
        for (int t = 0; t < s; ++t) { sc[t] = exp(sc[t] - mx); sum += sc[t]; }
        for (int t = 0; t < s; ++t) sc[t] = (double)(float)(sc[t] / sum);   /* weights stored fp32 */
        if (w_out) for (int t = 0; t < s; ++t) w_out[(size_t)hq * s + t] = (float)sc[t];
        for (int i = 0; i < Dh; ++i) {
            double acc = 0.0;
            for (int t = 0; t < s; ++t) {
                int32_t pg = bt_row[t / page];
                const uint16_t *vr = v_pool + (((size_t)pg * Hkv + hk) * page + (size_t)(t % page)) * Dh;
                acc += sc[t] * (double)orc_bf16_to_f32(vr[i]);
            }
            o[(size_t)hq * Dh + i] = (float)acc;
        }
    }
    free(sc);
    return 0;
}

/* ---- a8: silu(z) = z / (1 + exp(-z)) ------------------------------------------------------ */
float orc_silu(float z) { return (float)((double)z / (1.0 + exp(-(double)z))); }

/* ---- a11: replica copy = byte copy ("only memory copies") ------------------- */
void orc_replica_copy(void *dst, const void *src, size_t bytes) { memcpy(dst, src, bytes); }

/* ---- one sub-batch through one replica's weights ------------------------------------------ *
 * rows[0..M): original row indices (increasing).  hidden_in/out, pools, bt, seq_lens are the  *
 * full-batch arrays.  Rows with seq_lens <= 0 are left untouched (padding rows).               */
static int orc_sub_batch(const orc_desc *D, const orc_weights *W, const int32_t *rows, int M,
                         const uint16_t *hidden_in, uint16_t *hidden_out, uint16_t *k_pool,
                         uint16_t *v_pool, const int32_t *bt, int max_blocks, const int32_t *seq_lens,
                         const orc_taps *T) {
    const int d = D->hidden, Hq = D->n_q_heads, Hkv = D->n_kv_heads, Dh = D->head_dim, F = D->ffn;
    const int QD = Hq * Dh, KD = Hkv * Dh, page = D->page;
    if (M == 0) return 0;
    size_t Ms = (size_t)M;
    float *h = malloc(4 * Ms * d), *x = malloc(4 * Ms * d), *q = malloc(4 * Ms * QD);
    float *k = malloc(4 * Ms * KD), *v = malloc(4 * Ms * KD), *o = malloc(4 * Ms * QD);
    float *t0 = malloc(4 * Ms * d), *h1 = malloc(4 * Ms * d), *y = malloc(4 * Ms * d);
    float *gt = malloc(4 * Ms * F), *up = malloc(4 * Ms * F), *a = malloc(4 * Ms * F);
    float *dn = malloc(4 * Ms * d);
    int rc = 0;
    if (!h || !x || !q || !k || !v || !o || !t0 || !h1 || !y || !gt || !up || !a || !dn) { rc = -1; goto done; }

    for (int m = 0; m < M; ++m)
        for (int i = 0; i < d; ++i) h[Ms * 0 + (size_t)m * d + i] = orc_bf16_to_f32(hidden_in[(size_t)rows[m] * d + i]);

    orc_rmsnorm(h, W->g1, M, d, D->rms_eps, x);                                   /* a1 */
    orc_matmul_wt(x, W->wq, M, d, QD, q);                                        /* a2 */
    orc_matmul_wt(x, W->wk, M, d, KD, k);
    orc_matmul_wt(x, W->wv, M, d, KD, v);
    for (int m = 0; m < M; ++m) {
        int b = rows[m], s = seq_lens[b], p = s - 1;
        orc_rope(q + (size_t)m * QD, Hq, Dh, p, D->rope_base);                   /* a3 */
        orc_rope(k + (size_t)m * KD, Hkv, Dh, p, D->rope_base);
        int32_t pg = bt[(size_t)b * max_blocks + p / page];                      /* a4 */
        if (pg < 0) { rc = -2; goto done; }
        for (int hk = 0; hk < Hkv; ++hk)
            for (int i = 0; i < Dh; ++i) {
                size_t slot = (((size_t)pg * Hkv + hk) * page + (size_t)(p % page)) * Dh + i;
                k_pool[slot] = orc_f32_to_bf16(k[(size_t)m * KD + hk * Dh + i]);
                v_pool[slot] = orc_f32_to_bf16(v[(size_t)m * KD + hk * Dh + i]);
            }
    }
    {
        int arc = 0;
#pragma omp parallel for schedule(dynamic, 1)
        for (int m = 0; m < M; ++m) {                                            /* a5 */
            int b = rows[m];
            int r1 = orc_attention_decode(q + (size_t)m * QD, k_pool, v_pool, bt + (size_t)b * max_blocks,
                                          seq_lens[b], Hq, Hkv, Dh, page, o + (size_t)m * QD, NULL);
            if (r1) {
#pragma omp atomic write
                arc = r1;
            }
        }
        if (arc) { rc = arc; goto done; }
    }
    orc_matmul_wt(o, W->wo, M, QD, d, t0);                                       /* a6 */
    for (size_t i = 0; i < Ms * d; ++i) h1[i] = h[i] + t0[i];
    orc_rmsnorm(h1, W->g2, M, d, D->rms_eps, y);                                  /* a7 */
    orc_matmul_wt(y, W->wgate, M, d, F, gt);                                     /* a8 */
    orc_matmul_wt(y, W->wup, M, d, F, up);
    for (size_t i = 0; i < Ms * F; ++i) a[i] = orc_silu(gt[i]) * up[i];
    orc_matmul_wt(a, W->wdown, M, F, d, dn);                                     /* a9 */
    for (int m = 0; m < M; ++m) {
        int b = rows[m];
        for (int i = 0; i < d; ++i) {
            float r = h1[(size_t)m * d + i] + dn[(size_t)m * d + i];
            hidden_out[(size_t)b * d + i] = orc_f32_to_bf16(r);                  /* row b: original order */
            if (T && T->out) T->out[(size_t)b * d + i] = r;
        }
        if (T) {
            if (T->x) memcpy(T->x + (size_t)b * d, x + (size_t)m * d, 4 * (size_t)d);
            if (T->q) memcpy(T->q + (size_t)b * QD, q + (size_t)m * QD, 4 * (size_t)QD);
            if (T->k_new) memcpy(T->k_new + (size_t)b * KD, k + (size_t)m * KD, 4 * (size_t)KD);
            if (T->v_new) memcpy(T->v_new + (size_t)b * KD, v + (size_t)m * KD, 4 * (size_t)KD);
            if (T->o) memcpy(T->o + (size_t)b * QD, o + (size_t)m * QD, 4 * (size_t)QD);
            if (T->h1) memcpy(T->h1 + (size_t)b * d, h1 + (size_t)m * d, 4 * (size_t)d);
            if (T->y) memcpy(T->y + (size_t)b * d, y + (size_t)m * d, 4 * (size_t)d);
            if (T->a) memcpy(T->a + (size_t)b * F, a + (size_t)m * F, 4 * (size_t)F);
        }
    }
done:
    free(h); free(x); free(q); free(k); free(v); free(o); free(t0); free(h1); free(y);
    free(gt); free(up); free(a); free(dn);
    return rc;
}

static uint16_t *orc_dup(const uint16_t *src, size_t n) {
    uint16_t *p = (uint16_t *)malloc(2 * n);
    if (p) orc_replica_copy(p, src, 2 * n);
    return p;
}

/* ---- the replicated layer forward (SURVEY.md 8(c) pseudo-code) ------------------------------ *
 * hidden_in/out: bf16 [B][d] (may alias).  replica_assign[b] in [0, R).  Replica r > 0 runs     *
 * against ITS OWN byte copy of the weights (made here with orc_replica_copy), replica 0 against *
 * the originals.  Returns 0, or <0 on malloc failure / bad block table / bad assignment.        */
int orc_layer_forward(const orc_desc *D, const orc_weights *W, const uint16_t *hidden_in,
                      uint16_t *hidden_out, uint16_t *k_pool, uint16_t *v_pool, const int32_t *bt,
                      int max_blocks, const int32_t *seq_lens, const int32_t *replica_assign, int B,
                      int R, const orc_taps *T) {
    const size_t d = (size_t)D->hidden, QD = (size_t)D->n_q_heads * D->head_dim,
                 KD = (size_t)D->n_kv_heads * D->head_dim, F = (size_t)D->ffn;
    int rc = 0;
    int32_t *rows = (int32_t *)malloc(sizeof(int32_t) * (size_t)(B > 0 ? B : 1));
    uint16_t *in_copy = orc_dup(hidden_in, (size_t)B * d);     /* so that in/out may alias */
    if (!rows || !in_copy) { free(rows); free(in_copy); return -1; }
    if (hidden_out != hidden_in) memcpy(hidden_out, hidden_in, 2 * (size_t)B * d); /* padding rows pass through */
    for (int b = 0; b < B; ++b)
        if (seq_lens[b] > 0 && (replica_assign[b] < 0 || replica_assign[b] >= R)) { rc = -3; goto done; }
    for (int r = 0; r < R && rc == 0; ++r) {                   /* replica loop: PAPER.md:93, 101 */
        int M = 0;
        for (int b = 0; b < B; ++b)
            if (replica_assign[b] == r && seq_lens[b] > 0) rows[M++] = b;   /* stable, increasing b */
        if (M == 0) continue;                                   /* empty group is legal: PAPER.md:217 */
        if (r == 0) {
            rc = orc_sub_batch(D, W, rows, M, in_copy, hidden_out, k_pool, v_pool, bt, max_blocks, seq_lens, T);
        } else {
            orc_weights Wr;                                     /* replica = byte copy: PAPER.md:91 */
            uint16_t *c[9];
            c[0] = orc_dup(W->g1, d);        c[1] = orc_dup(W->wq, QD * d);   c[2] = orc_dup(W->wk, KD * d);
            c[3] = orc_dup(W->wv, KD * d);   c[4] = orc_dup(W->wo, d * QD);   c[5] = orc_dup(W->g2, d);
            c[6] = orc_dup(W->wgate, F * d); c[7] = orc_dup(W->wup, F * d);   c[8] = orc_dup(W->wdown, d * F);
            int ok = 1;
            for (int i = 0; i < 9; ++i) ok = ok && c[i];
            if (ok) {
                Wr.g1 = c[0]; Wr.wq = c[1]; Wr.wk = c[2]; Wr.wv = c[3]; Wr.wo = c[4];
                Wr.g2 = c[5]; Wr.wgate = c[6]; Wr.wup = c[7]; Wr.wdown = c[8];
                rc = orc_sub_batch(D, &Wr, rows, M, in_copy, hidden_out, k_pool, v_pool, bt, max_blocks, seq_lens, T);
            } else rc = -1;
            for (int i = 0; i < 9; ++i) free(c[i]);
        }
    }
done:
    free(rows); free(in_copy);
    return rc;
}

/* ---- a0: micro-batch grouping (stable partition by replica; exact integers) ------------------ *
 * perm[pos] = original row, rows of replica 0 first (increasing b), then replica 1, ...;        *
 * counts[r] = rows of replica r.  Rows with seq_lens <= 0 are dropped.  Returns rows kept.      */
int orc_group_rows(const int32_t *replica_assign, const int32_t *seq_lens, int B, int R,
                   int32_t *perm, int32_t *counts) {
    int n = 0;
    for (int r = 0; r < R; ++r) {
        counts[r] = 0;
        for (int b = 0; b < B; ++b)
            if (seq_lens[b] > 0 && replica_assign[b] == r) { perm[n++] = b; counts[r]++; }
    }
    return n;
}

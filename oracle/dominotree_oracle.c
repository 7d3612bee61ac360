/*
 * dominotree_oracle.c -- TEST INFRASTRUCTURE ONLY.
 *
 * A plain, slow, float64 CPU statement of DominoTree's per-round draft-tree builder
 * (arxiv/paper_2607_08642), written from the paper and used ONLY by tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg.  It shares no
 * code, header, table or helper with the CUDA path (paper_2607_08642_b200/csrc) and the
 * product never calls it.
 *
 * What it computes (citations are /root/reference/PAPER.md line numbers):
 *   - top-M marginal candidates per depth                       PAPER.md:133, 141 (Alg. 1 step 1)
 *   - Domino's causal encoder, a single-layer no-bias GRU       PAPER.md:68-72   (Sec. 2.3)
 *   - Domino's correction head dL = W2 SiLU(W1 [H; S])          PAPER.md:74-78   (Sec. 2.3)
 *   - CHILDREN(S, d): corrected log-probabilities restricted
 *     to the depth-d top-M slice, top-k of them                 PAPER.md:142-144 (Alg. 1 step 2)
 *   - best-first expansion to node budget n (=B)                PAPER.md:145-149 (Alg. 1 steps 3-5)
 *   - ancestor-only tree-attention mask, positions
 *
 * Readings of the paper where it is silent:
 *   A1  log-probability = log-softmax over the M-slice of (base logit + dL)/T_eff.
 *   A2  GRU = PyTorch nn.GRU convention: rows of W_ih/W_hh stacked (r, z, n),
 *       n = tanh(W_in x + r*(W_hn h)), h' = (1-z)*n + z*h, no biases.
 *   A4  S_0 = GRUcell(h=0, x=E[root token]).
 *   A7  T_eff = 1 if temperature == 0 else temperature; divides (base + dL).
 *   A8  every ordering is (score desc, token id asc), completed by (parent slot asc) in the heap.
 *   A9  loop while |T| < B and heap non-empty; depth only gates expansion (d < L).
 *   A10 slot 0 = root; dead leaf = token 0, parent 0, depth 1, score -inf, mask {root, self}.
 *   PARITY UNPINNED by the paper for the numeric conventions A1, A2, A4 (no worked example is
 *   printed and the released checkpoint/code is absent); everything else is pinned by
 *   tests/test_oracle_pins.py (library routines, DDTree reduction, chain reduction, brute force).
 *
 * One deviation in evaluation ORDER only (not in values): Alg. 1 returns each child's advanced
 * GRU state from CHILDREN; a child's state is a pure function of (parent state,
 * child token), so by default it is evaluated when the child is popped.  eager_states=1 follows
 * the paper's order literally; tests assert both give bit-identical output.
 *
 * The heap is a linear scan for the maximum -- no blocking, fusion or reordering.
 * All arithmetic is IEEE double; inputs are widened exactly from bf16 / fp32.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

enum { ORC_BF16 = 0, ORC_F32 = 1, ORC_F64 = 2 };

typedef struct {
    const void *embed;   /* E    [V, d] */
    const void *w_ih;    /* W_ih [3g, d]  rows r,z,n */
    const void *w_hh;    /* W_hh [3g, g]                                             */
    const void *w1;      /* W1   [r, d+g] cols [0,d) on H, [d,d+g) on S */
    const void *w2;      /* W2   [V, r] */
    int32_t V, d, g, r;
    int32_t dtype;       /* ORC_BF16 | ORC_F32 | ORC_F64, for all five and for logits/hidden */
} orc_weights;

static inline double ldv(const void *p, size_t i, int dt) {
    if (dt == ORC_BF16) {
        uint32_t u = ((uint32_t)((const uint16_t *)p)[i]) << 16;
        float f;
        memcpy(&f, &u, 4);
        return (double)f;
    }
    if (dt == ORC_F32) return (double)((const float *)p)[i];
    return ((const double *)p)[i];
}

static double sigmoid(double x) { return 1.0 / (1.0 + exp(-x)); }
static double silu(double x) { return x * sigmoid(x); }   /* SiLU(x) = x*sigma(x) */

/* ---------------------------------------------------------------- top-M select (Alg. 1 step 1) */
typedef struct { double v; int32_t i; } orc_pair;

static int cmp_pair_desc(const void *a, const void *b) {
    const orc_pair *x = (const orc_pair *)a, *y = (const orc_pair *)b;
    if (x->v > y->v) return -1;
    if (x->v < y->v) return 1;
    return (x->i > y->i) - (x->i < y->i);   /* tie: lower token id first (A8) */
}

/* ids/vals of the M largest entries of one row, ordered (value desc, token asc). */
int orc_select_topm(const void *row, int32_t dtype, int32_t V, int32_t M, int32_t *ids, double *vals) {
    if (M < 1 || M > V) return -1;
    orc_pair *p = (orc_pair *)malloc(sizeof(orc_pair) * (size_t)V);
    if (!p) return -2;
    for (int32_t t = 0; t < V; ++t) { p[t].v = ldv(row, (size_t)t, dtype); p[t].i = t; }
    qsort(p, (size_t)V, sizeof(orc_pair), cmp_pair_desc);
    for (int32_t m = 0; m < M; ++m) { ids[m] = p[m].i; vals[m] = p[m].v; }
    free(p);
    return 0;
}

/* ---------------------------------------------------------------- GRU cell (Sec. 2.3, A2) */
/* h_out = GRUcell(h, x = E[token]); h, h_out have g entries. */
int orc_gru_cell(const orc_weights *w, const double *h, int32_t token, double *h_out) {
    const int d = w->d, g = w->g, dt = w->dtype;
    if (token < 0 || token >= w->V) return -1;
    const size_t xoff = (size_t)token * (size_t)d;
    for (int j = 0; j < g; ++j) {
        double ir = 0, iz = 0, in = 0, hr = 0, hz = 0, hn = 0;
        for (int c = 0; c < d; ++c) {
            double x = ldv(w->embed, xoff + c, dt);
            ir += ldv(w->w_ih, (size_t)(0 * g + j) * d + c, dt) * x;
            iz += ldv(w->w_ih, (size_t)(1 * g + j) * d + c, dt) * x;
            in += ldv(w->w_ih, (size_t)(2 * g + j) * d + c, dt) * x;
        }
        for (int c = 0; c < g; ++c) {
            double s = h[c];
            hr += ldv(w->w_hh, (size_t)(0 * g + j) * g + c, dt) * s;
            hz += ldv(w->w_hh, (size_t)(1 * g + j) * g + c, dt) * s;
            hn += ldv(w->w_hh, (size_t)(2 * g + j) * g + c, dt) * s;
        }
        double rg = sigmoid(ir + hr);
        double zg = sigmoid(iz + hz);
        double ng = tanh(in + rg * hn);
        h_out[j] = (1.0 - zg) * ng + zg * h[j];
    }
    return 0;
}

/* ---------------------------------------------------------------- correction + slice log-softmax */
/* logp[m] for all m < M: log-softmax over the slice of (base[m] + W2[cand[m],:] . a) / T_eff,
   a = SiLU(W1 [H_i; S]).  PAPER.md:76, 143-144; readings A1, A7. */
int orc_slice_logprobs(const orc_weights *w, const void *H_i /* d values, w->dtype */, const double *S,
                       const int32_t *cand, const double *base, int32_t M, double T_eff, double *logp) {
    const int d = w->d, g = w->g, r = w->r, dt = w->dtype;
    double *a = (double *)malloc(sizeof(double) * (size_t)r);
    if (!a) return -2;
    for (int j = 0; j < r; ++j) {
        double acc = 0;
        for (int c = 0; c < d; ++c) acc += ldv(w->w1, (size_t)j * (d + g) + c, dt) * ldv(H_i, (size_t)c, dt);
        for (int c = 0; c < g; ++c) acc += ldv(w->w1, (size_t)j * (d + g) + d + c, dt) * S[c];
        a[j] = silu(acc);
    }
    double zmax = -INFINITY;
    for (int m = 0; m < M; ++m) {
        double dl = 0;
        for (int j = 0; j < r; ++j) dl += ldv(w->w2, (size_t)cand[m] * r + j, dt) * a[j];
        logp[m] = (base[m] + dl) / T_eff;            /* holds z_m for now */
        if (logp[m] > zmax) zmax = logp[m];
    }
    double sum = 0;
    for (int m = 0; m < M; ++m) sum += exp(logp[m] - zmax);
    double lse = zmax + log(sum);
    for (int m = 0; m < M; ++m) logp[m] -= lse;
    free(a);
    return 0;
}

/* CHILDREN(S, i) of Alg. 1 step 2: the k best slice entries by (logp desc, token asc). */
int orc_children(const orc_weights *w, const void *H_i, const double *S, const int32_t *cand,
                 const double *base, int32_t M, int32_t k, double T_eff,
                 int32_t *out_tok, double *out_logp, double *all_logp /* M, may be NULL */) {
    if (k < 1 || k > M) return -1;
    double *lp = (double *)malloc(sizeof(double) * (size_t)M);
    orc_pair *p = (orc_pair *)malloc(sizeof(orc_pair) * (size_t)M);
    if (!lp || !p) { free(lp); free(p); return -2; }
    int rc = orc_slice_logprobs(w, H_i, S, cand, base, M, T_eff, lp);
    if (rc) { free(lp); free(p); return rc; }
    for (int m = 0; m < M; ++m) { p[m].v = lp[m]; p[m].i = cand[m]; }
    qsort(p, (size_t)M, sizeof(orc_pair), cmp_pair_desc);
    for (int c = 0; c < k; ++c) { out_tok[c] = p[c].i; out_logp[c] = p[c].v; }
    if (all_logp) memcpy(all_logp, lp, sizeof(double) * (size_t)M);
    free(lp); free(p);
    return 0;
}

/* ---------------------------------------------------------------- Algorithm 1 */
typedef struct {
    int32_t token, parent, depth;
    double g;          /* cumulative corrected log-score */
    double *state;     /* only with eager_states */
} orc_entry;

/* (g desc, token asc, parent slot asc) -- A8 */
static int entry_better(const orc_entry *x, const orc_entry *y) {
    if (x->g != y->g) return x->g > y->g;
    if (x->token != y->token) return x->token < y->token;
    return x->parent < y->parent;
}

/*
 * One request.  logits [L, V], hidden [L, d] in w->dtype.  N = B+1 output slots.
 * Outputs (caller-allocated): tokens, parents, depths, positions [N] i32; scores [N] f64;
 * mask [N*N] u8; n_nodes [1]; cand_ids [L*M] i32, cand_vals [L*M] f64 (the select result);
 * residual heap (entries never popped): res_token/parent/depth [B*k] i32, res_score [B*k] f64,
 * n_res [1].  Returns 0, or <0 on bad arguments / allocation failure.
 */
int orc_build_tree(const orc_weights *w, const void *logits, const void *hidden, int32_t L,
                   int32_t root_token, int32_t root_pos, int32_t M, int32_t B, int32_t k,
                   double temperature, int32_t eager_states,
                   int32_t *tokens, int32_t *parents, int32_t *depths, int32_t *positions,
                   double *scores, uint8_t *mask, int32_t *n_nodes,
                   int32_t *cand_ids, double *cand_vals,
                   int32_t *res_token, int32_t *res_parent, int32_t *res_depth, double *res_score,
                   int32_t *n_res) {
    const int V = w->V, d = w->d, g = w->g, dt = w->dtype;
    if (L < 1 || M < 1 || M > V || k < 1 || k > M || B < 1 || temperature < 0 || !(temperature == temperature))
        return -1;
    if (root_token < 0 || root_token >= V) return -1;
    const int N = B + 1;
    const double T_eff = (temperature == 0.0) ? 1.0 : temperature;           /* step 1, A7 */
    const size_t esz = (dt == ORC_BF16) ? 2 : (dt == ORC_F32 ? 4 : 8);

    /* step 2: per-depth top-M */
    for (int i = 0; i < L; ++i) {
        int rc = orc_select_topm((const char *)logits + (size_t)i * V * esz, dt, V, M,
                                 cand_ids + (size_t)i * M, cand_vals + (size_t)i * M);
        if (rc) return rc;
    }

    size_t cap = (size_t)B * (size_t)k + (size_t)k;
    orc_entry *heap = (orc_entry *)calloc(cap, sizeof(orc_entry));
    double *states = (double *)calloc((size_t)N * g, sizeof(double));    /* state of slot s */
    double *zero = (double *)calloc((size_t)g, sizeof(double));
    int32_t *ctok = (int32_t *)malloc(sizeof(int32_t) * (size_t)k);
    double *clp = (double *)malloc(sizeof(double) * (size_t)k);
    if (!heap || !states || !zero || !ctok || !clp) { free(heap); free(states); free(zero); free(ctok); free(clp); return -2; }
    size_t hn = 0;
    int rc = 0;

    /* step 3: S_0 = GRUcell(0, E[root])  (A4) */
    rc = orc_gru_cell(w, zero, root_token, states);
    tokens[0] = root_token; parents[0] = -1; depths[0] = 0; scores[0] = 0.0;
    int n = 0;

    /* step 5 (Alg. 1 step 3): heap <- CHILDREN(S_0, 1); then step 6 (Alg. 1 step 4) loop */
    int expand_slot = 0;   /* slot whose children are pushed next; -1 = none */
    while (rc == 0) {
        if (expand_slot >= 0) {
            int dep = depths[expand_slot];                 /* children live at depth dep+1 */
            const void *H_i = (const char *)hidden + (size_t)dep * d * esz;       /* H_{dep+1}: row index dep (A12) */
            rc = orc_children(w, H_i, states + (size_t)expand_slot * g,
                              cand_ids + (size_t)dep * M, cand_vals + (size_t)dep * M, M, k, T_eff,
                              ctok, clp, NULL);
            if (rc) break;
            for (int c = 0; c < k; ++c) {
                orc_entry e;
                e.token = ctok[c]; e.parent = expand_slot; e.depth = dep + 1;
                e.g = scores[expand_slot] + clp[c];
                e.state = NULL;
                if (eager_states) {                        /* state advanced per child */
                    e.state = (double *)malloc(sizeof(double) * (size_t)g);
                    if (!e.state) { rc = -2; break; }
                    rc = orc_gru_cell(w, states + (size_t)expand_slot * g, e.token, e.state);
                    if (rc) break;
                }
                heap[hn++] = e;
            }
            if (rc) break;
        }
        if (n >= B || hn == 0) break;
        /* pop the maximal entry (linear scan) */
        size_t best = 0;
        for (size_t q = 1; q < hn; ++q) if (entry_better(&heap[q], &heap[best])) best = q;
        orc_entry e = heap[best];
        heap[best] = heap[hn - 1];
        --hn;
        ++n;
        tokens[n] = e.token; parents[n] = e.parent; depths[n] = e.depth; scores[n] = e.g;
        if (e.state) {
            memcpy(states + (size_t)n * g, e.state, sizeof(double) * (size_t)g);
            free(e.state);
        } else {
            rc = orc_gru_cell(w, states + (size_t)e.parent * g, e.token, states + (size_t)n * g);
            if (rc) break;
        }
        expand_slot = (e.depth < L) ? n : -1;   /* Alg. 1 step 4(b): if d < L push CHILDREN(S_d, d+1) */
    }

    /* step 7: emit */
    if (rc == 0) {
        *n_nodes = n + 1;
        for (int s = n + 1; s < N; ++s) { tokens[s] = 0; parents[s] = 0; depths[s] = 1; scores[s] = -INFINITY; }
        for (int s = 0; s < N; ++s) positions[s] = root_pos + depths[s];
        memset(mask, 0, (size_t)N * N);
        for (int s = 0; s < N; ++s) {
            int a = s;
            while (a >= 0) { mask[(size_t)s * N + a] = 1; a = parents[a]; }
        }
        *n_res = (int32_t)hn;
        for (size_t q = 0; q < hn; ++q) {
            res_token[q] = heap[q].token; res_parent[q] = heap[q].parent;
            res_depth[q] = heap[q].depth; res_score[q] = heap[q].g;
        }
    }
    for (size_t q = 0; q < hn; ++q) free(heap[q].state);
    free(heap); free(states); free(zero); free(ctok); free(clp);
    return rc;
}

/*
 * score_path: corrected log-probability of each token of a given path u_1..u_len under its own
 * prefix (the g(u) of Alg. 1), evaluated step by step with the same CHILDREN scorer.
 * cand_ids/cand_vals: the select result [L*M].  Outputs per level: logp[len] (NaN if the token is
 * not among the depth's M candidates), rank[len] = 0-based rank in the (logp desc, token asc)
 * order of the slice (-1 if absent), kth_logp[len] = the k-th best logp of that slice.
 */
int orc_score_path(const orc_weights *w, const void *hidden, int32_t L, int32_t root_token,
                   const int32_t *cand_ids, const double *cand_vals, int32_t M, int32_t k,
                   double temperature, const int32_t *path, int32_t len,
                   double *logp, int32_t *rank, double *kth_logp) {
    const int d = w->d, g = w->g, dt = w->dtype;
    if (len < 0 || len > L) return -1;
    const double T_eff = (temperature == 0.0) ? 1.0 : temperature;
    const size_t esz = (dt == ORC_BF16) ? 2 : (dt == ORC_F32 ? 4 : 8);
    double *S = (double *)calloc((size_t)g, sizeof(double));
    double *S2 = (double *)calloc((size_t)g, sizeof(double));
    double *lp = (double *)malloc(sizeof(double) * (size_t)M);
    int32_t *ct = (int32_t *)malloc(sizeof(int32_t) * (size_t)k);
    double *cl = (double *)malloc(sizeof(double) * (size_t)k);
    if (!S || !S2 || !lp || !ct || !cl) { free(S); free(S2); free(lp); free(ct); free(cl); return -2; }
    int rc = orc_gru_cell(w, S2, root_token, S);     /* S_0 from h = 0 (S2 is zero here) */
    for (int i = 0; i < len && rc == 0; ++i) {
        const int32_t *cand = cand_ids + (size_t)i * M;
        rc = orc_children(w, (const char *)hidden + (size_t)i * d * esz, S, cand,
                          cand_vals + (size_t)i * M, M, k, T_eff, ct, cl, lp);
        if (rc) break;
        kth_logp[i] = cl[k - 1];
        int pos = -1;
        for (int m = 0; m < M; ++m) if (cand[m] == path[i]) { pos = m; break; }
        if (pos < 0) { logp[i] = NAN; rank[i] = -1; }
        else {
            logp[i] = lp[pos];
            int rk = 0;
            for (int m = 0; m < M; ++m)
                if (lp[m] > lp[pos] || (lp[m] == lp[pos] && cand[m] < cand[pos])) ++rk;
            rank[i] = rk;
        }
        rc = orc_gru_cell(w, S, path[i], S2);
        memcpy(S, S2, sizeof(double) * (size_t)g);
    }
    free(S); free(S2); free(lp); free(ct); free(cl);
    return rc;
}

int orc_version(void) { return 1; }

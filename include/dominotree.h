/*
 * dominotree.h -- C-ABI boundary of the B200-native DominoTree per-round draft-tree builder.
 *
 * The operation is Algorithm 1 of the paper (Sec. 3.2 "DominoTree builder"):
 * per request and decoding round, (1) take the drafter's L x V marginal logits L_i^base
 * (PAPER.md:56-62), (2) select the top-M candidate tokens at each block position
 * (PAPER.md:133, 141), (3) run the best-first max-heap expansion to node budget B
 * (PAPER.md:93, 109, 145-148), scoring the children of each popped node with Domino's
 * path-dependent correction  L_i = L_i^base + W2 SiLU(W1 [H_i; S_{i-1}]),  S_{i-1} = GRU(E_{<=i-1})
 * restricted to the M candidates, and (4) emit the
 * tree tokens, parents, depths, positions and the ancestor-only tree-attention mask for the
 * verifier.  Readings of the paper where it is silent are listed in
 * DESIGN.md ("Readings"): slice log-softmax (A1), PyTorch GRU gate convention (A2),
 * S_0 = GRUcell(0, E[root]) (A4), T_eff (A7), tie-breaks (A8), dead-leaf padding (A10).
 *
 * Everything below runs in hand-written sm_100a CUDA kernels inside libdominotree.so; there is
 * no CPU fallback.  No torch types cross this boundary: plain pointers and sizes only.
 *
 * Pointer convention: every data pointer is a DEVICE pointer owned by the caller and borrowed
 * for the stream-ordered duration of the call (weights: for the lifetime of the handle).  The
 * only host pointers are the handle, the dt_weights / dt_outputs structs themselves (read
 * synchronously during the call) and the `_host` entry point, which says so in its name.
 *
 * Error behaviour: every entry point returns DT_OK (0) or a negative dt_status; nothing throws,
 * aborts or prints.  On error no output buffer content is defined.
 */
#ifndef DOMINOTREE_H
#define DOMINOTREE_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct dt_handle dt_handle;

/* dtype of marginal_logits, backbone_hidden and all five weight tensors (one dtype for all). */
typedef enum { DT_BF16 = 0, DT_F32 = 1 } dt_dtype;

typedef enum {
    DT_OK = 0,
    DT_ERR_INVALID_ARG = -1, /* null pointer, shape/parameter out of range                       */
    DT_ERR_UNSUPPORTED = -2, /* shape beyond the compiled limits (see DT_MAX_*)                  */
    DT_ERR_CUDA = -3,        /* a CUDA runtime call failed (dt_last_cuda_error gives the code)   */
    DT_ERR_ALLOC = -4,       /* device or host allocation failed                                 */
    DT_ERR_STATIC_LIMIT = -5 /* dt_select_topm_static: shape beyond its static scratch limits    */
} dt_status;

/* compiled limits */
#define DT_MAX_M 256   /* candidate width                                   */
#define DT_MAX_B 255   /* node budget (N = B+1 <= 256 output slots)         */
#define DT_MAX_K 32    /* branching factor                                  */
#define DT_MAX_L 64    /* block depth                                       */

/* Frozen drafter weights.  Row-major, dense, no biases. */
typedef struct {
    const void *embed;    /* E    [V, d]     frozen target token embedding    */
    const void *gru_w_ih; /* W_ih [3g, d]    rows stacked (r, z, n) gates (reading A2) PAPER.md:68   */
    const void *gru_w_hh; /* W_hh [3g, g]                                                            */
    const void *corr_w1;  /* W1   [r, d+g]   cols [0,d) act on H_i, [d,d+g) on S_{i-1} PAPER.md:76   */
    const void *corr_w2;  /* W2   [V, r]     rank-r -> vocabulary projection*/
    int32_t V, d, g, r;
    int32_t dtype;        /* dt_dtype */
} dt_weights;

/* Caller-allocated device outputs; N = B+1 slots per request, slot 0 = the root (reading A10).
 * All are fully overwritten for `batch` requests, padding slots included. */
typedef struct {
    int32_t *tokens;    /* [batch, N]    tokens[b,0] = root_tokens[b]; slots 1.. in pop order */
    int32_t *parents;   /* [batch, N]    parent slot; -1 for the root; parents[b,i] < i        */
    int32_t *depths;    /* [batch, N]    0 for the root, 1..L                                                 */
    int32_t *positions; /* [batch, N]    root_positions[b] + depth (0-based if root_positions is NULL)        */
    float *scores;      /* [batch, N]    cumulative corrected log-score g(u); 0 for the root   */
    uint8_t *mask;      /* [batch, N, N] mask[b,i,j] = 1 iff j == i or j is an ancestor of i*/
    int32_t *n_nodes;   /* [batch]       valid slots incl. root; slots >= n_nodes are dead leaves:            */
                        /*               token 0, parent 0, depth 1, score -inf, mask row {root, self}        */
} dt_outputs;

/*
 * dt_create: validate shapes, allocate the per-handle device workspace for up to `max_batch`
 * requests of block depth L, candidate width <= max_M, budget <= max_B and branching factor k
 * (paper: k = 8), and build the weight-only table P = E W_ih^T  [V, 3g] fp32
 * (the input half of every GRU step, becomes a row gather).  Synchronises the
 * device; not capture-safe.  Weights are borrowed until dt_destroy.
 * Errors: INVALID_ARG for null pointers or !(1 <= k <= max_M <= V), !(1 <= max_B), L < 1,
 * max_batch < 1, V/d/g/r < 1; UNSUPPORTED beyond DT_MAX_*; ALLOC; CUDA.
 */
int dt_create(dt_handle **h, const dt_weights *w, int32_t max_batch, int32_t L,
              int32_t max_M, int32_t max_B, int32_t k);

/*
 * dt_build_trees: one tree-build round (Algorithm 1) for `batch` independent
 * requests.
 *   marginal_logits  [batch, L, V]  device, handle dtype  -- L_i^base
 *   backbone_hidden  [batch, L, d]  device, handle dtype  -- H_i; row i-1 pairs with
 *                                                            parent state S_{i-1}
 *   root_tokens      [batch] int32  device                -- the verified token x_t
 *   root_positions   [batch] int32  device or NULL
 *   M in [k, max_M], B in [1, max_B], temperature >= 0 finite (0 means T_eff = 1, reading A7)
 * Asynchronous and capture-safe: only enqueues work on `stream` (a cudaStream_t), never
 * allocates, never synchronises, takes no data-dependent host branch -- the caller may capture
 * the whole round into one CUDA graph.  One handle serves one stream at a time.
 * Input values are assumed non-NaN (-inf logits are allowed and sort last).
 */
/* (`stream` is a cudaStream_t passed as void * so that this header needs no CUDA header.) */
int dt_build_trees(dt_handle *h, const void *marginal_logits, const void *backbone_hidden,
                   const int32_t *root_tokens, const int32_t *root_positions, int32_t batch,
                   int32_t M, int32_t B, float temperature, const dt_outputs *out, void *stream);

/*
 * dt_select_topm: step 1 of Algorithm 1 alone: for each of `rows` rows of
 * `logits` [rows, V] (device, handle dtype) write the token ids and values of the M largest
 * entries, ordered (value desc, token id asc) with -0 == +0, to cand_id [rows, M] int32 and
 * cand_val [rows, M] float (device).  rows <= max_batch * L.  Asynchronous, capture-safe.
 */
int dt_select_topm(dt_handle *h, const void *logits, int32_t rows, int32_t M,
                   int32_t *cand_id, float *cand_val, void *stream);

/*
 * dt_select_topm_static: the same operation as dt_select_topm for callers that cannot
 * allocate: no handle, no cudaMalloc / cudaFree, no allocating library call, nothing to free.  The scratch
 * memory the select kernels need (per-row arrival tickets and thresholds, per-chunk partial lists) is ONE
 * file-scope device array of the library, 8 KiB + DT_STATIC_PART_BYTES (2 MiB) per GPU, held from the moment
 * the library is loaded on that GPU until exit.
 *   logits  [rows, V] device, element type `dtype` (DT_BF16 or DT_F32), row-major, contiguous
 *   cand_id [rows, M] int32 device, cand_val [rows, M] float device: outputs, caller-owned; same
 *           order as dt_select_topm: (value desc, token id asc), -0 == +0
 *   stream  a cudaStream_t (as void *) of the CURRENT device; the call only enqueues a memset node and one
 *           kernel on it (asynchronous)
 * Limits: rows <= DT_STATIC_MAX_ROWS (1024) and M <= DT_MAX_M, else DT_ERR_STATIC_LIMIT (nothing is
 * enqueued); rows < 0, V < 1, M < 1, M > V, a bad dtype or a null pointer with rows > 0: DT_ERR_INVALID_ARG;
 * rows == 0 is a no-op.  Sharing: every call on a GPU uses the same array, which keeps the previous call's
 * contents (what must start at zero is cleared on `stream` in front of the kernel): calls on one stream are
 * safe back to back, calls that OVERLAP on the GPU (two streams, concurrent graph replays) race and give
 * wrong candidates.  The first call on a device resolves the array's device address and sets kernel
 * attributes (once per device, that device current; thread-safe); dt_static_init() does that set-up for the
 * current device ahead of time, e.g. before a stream capture.
 */
#define DT_STATIC_MAX_ROWS 1024
#define DT_STATIC_PART_BYTES (2u << 20)
int dt_static_init(void);
int dt_select_topm_static(const void *logits, int32_t dtype, int32_t rows, int32_t V, int32_t M,
                          int32_t *cand_id, float *cand_val, void *stream);

/*
 * dt_build_trees_host: the same round with HOST buffers (pinned or pageable): copies the inputs
 * host->device, runs dt_build_trees, copies the outputs device->host and synchronises `stream`.
 * `out` members are HOST pointers here.  Uses staging buffers owned by the handle.
 * Not capture-safe (it synchronises).
 */
int dt_build_trees_host(dt_handle *h, const void *marginal_logits_host, const void *backbone_hidden_host,
                        const int32_t *root_tokens_host, const int32_t *root_positions_host,
                        int32_t batch, int32_t M, int32_t B, float temperature,
                        const dt_outputs *out_host, void *stream);

/*
 * dt_tree_links: first-child / next-sibling arrays of the trees of one round, for tree-verify kernels that walk the
 * tree instead of reading the mask (Sec. 3.5 verifies all nodes in one pass under the ancestor-only mask;
 * PAPER.md:187 runs the serving build on SGLang's EAGLE tree-verify kernel).  `tree` = the dt_outputs a dt_build_trees
 * call filled (device pointers; parents and n_nodes are read), B the budget of that call (N = B + 1 slots).  Outputs
 * (device, int32 [batch, N]): first_child[i] = the smallest slot j > i with parents[j] == i, next_sibling[i] = the
 * smallest slot j > i with parents[j] == parents[i]; -1 where there is none, for the root's sibling and for dead-leaf
 * padding slots.  Siblings are therefore chained in pop order (best first).  Asynchronous, capture-safe.
 * Errors: INVALID_ARG for null pointers, batch or B out of range.
 */
int dt_tree_links(dt_handle *h, const dt_outputs *tree, int32_t batch, int32_t B, int32_t *first_child,
                  int32_t *next_sibling, void *stream);

/*
 * dt_commit_paths: longest-accepted-path commit over the trees of one round (Sec. 3.5: "we
 * commit the highest-scoring root-to-leaf path along which every edge is accepted").  `tree` holds the DEVICE
 * outputs of dt_build_trees for the same batch and B (tokens, parents, depths, scores, n_nodes are read; N = B+1).
 * Exactly one of the two acceptance inputs is non-NULL:
 *   target_next [batch, N] int32 device -- greedy verification: the token the target model predicts after each
 *                tree node; the edge parent u -> node i is accepted iff tokens[i] == target_next[u];
 *   edge_ok     [batch, N] uint8 device -- any other rule: edge into node i accepted iff edge_ok[i] != 0.
 * A node is reachable iff every edge of its root path is accepted; the path ends at the reachable node of greatest
 * depth, then highest draft score, then lowest slot (dead-leaf padding slots never qualify).  Outputs (device):
 *   accept_len  [batch]        number of accepted draft tokens (depth of the end node, 0 = only the root)
 *   path_slots  [batch, L+1]   tree slots of the path, root first, padded with -1
 *   bonus_token [batch] or NULL  target_next at the end node (-1 in edge_ok mode)
 * Asynchronous, capture-safe.  Errors: INVALID_ARG for null pointers, both or neither acceptance input, batch or B
 * out of range.
 */
int dt_commit_paths(dt_handle *h, const dt_outputs *tree, int32_t batch, int32_t B, const int32_t *target_next,
                    const uint8_t *edge_ok, int32_t *accept_len, int32_t *path_slots, int32_t *bonus_token, void *stream);

/*
 * dt_adaptive_budget: CaDDTree's cost-aware stopping rule on the pop order of the built trees (PAPER.md:97-101,
 * 161-165): theta(n) = (1 + Phi(n)) / (C_d + C_v(n)), Phi(n) = sum over slots 1..n of exp(scores); n_star is the
 * first n with theta(n + 1) <= theta(n) (or every valid draft node).  `tree` = DEVICE outputs of dt_build_trees for
 * the same batch and B (scores, n_nodes are read); cv [B + 1] float device = verification cost of an n-node tree,
 * C_d = draft cost (same unit).  Outputs (device): n_star [batch] int32 draft nodes to keep (slots 1..n_star),
 * phi [batch] float or NULL = Phi(n_star).  The paper reports the rule as a negative result on the corrected tree
 * (it runs to the cap); it is provided as the measurement device of that claim.  Asynchronous, capture-safe.
 */
int dt_adaptive_budget(dt_handle *h, const dt_outputs *tree, int32_t batch, int32_t B, double C_d, const float *cv,
                       int32_t *n_star, float *phi, void *stream);

/* dt_set_option: knobs; unknown name or value -> INVALID_ARG.
 *   "scorer"        children function of dt_build_trees, the three arms of PAPER.md:553-555 (Appendix D):
 *                   0 DominoTree (Alg. 1, per-node path-dependent correction; default),
 *                   1 Marg (base logits alone, one menu per depth, no GRU),
 *                   2 Cond-static (correction once per depth along Domino's greedy chain, menu shared per depth;
 *                     bf16 shapes the fused kernel accepts, else dt_build_trees returns DT_ERR_UNSUPPORTED);
 *   "schedule"      0 best-first heap (Algorithm 1; default), 1 the frontier builder of the paper's serving path
 *                    with W = B: the same tree on tie-free inputs (bf16 shapes: the wavefront
 *                   kernel at its maximal width; fp32 and odd shapes: depth-synchronous ledger kernels);
 *   "adaptive_schedule"  1 (default): per round the device picks, from the mean top-1 probability of the base slices,
 *                   the wavefront kernel (bushy trees) or the lock-step kernel (chains); both give the same tree, scores
 *                   agree to fp32 rounding.  0: always the wavefront kernel when the shape allows (bitwise batch
 *                   invariance of the scores then holds for any mix of requests);
 *   "wave_width"    nodes a request may expand per dependent step of the wavefront kernel (0 = auto, 1 = the plain heap
 *                   schedule, up to 15); any value gives the same tree;
 *   "expand_path"   0 auto, 1 per-step kernels, 2 / 3 lock-step kernel on mma.sync, 4 lock-step kernel on tcgen05,
 *                   5 wavefront kernel;
 *   "select_chunks", "select_kernel", "select_span", "precompute_gemm", "precompute_serial"   tuning / measurement
 *   "lockstep_speculation"  lock-step kernel: the GRU CTAs run the pass of the node a chain would pop next while the
 *                     request CTA still scores its parent (or the frontier entry the request CTA hints at).  1 (default):
 *                     whenever the batch fits one request group (<= 32) on tcgen05 shapes with V <= 2^24, DominoTree
 *                     scorer; 2: also with several groups and for the Cond-static arm; 0: never.
 *                     Changes when a node's state is computed, never the result (bit-identical outputs).
 *   "lockstep_group"  lock-step kernel: requests per GRU pass (0 = automatic)
 *                   switches of the kernels.
 * Batch sizes: any batch <= max_batch runs on the persistent kernels (bf16): a launch of the wavefront kernel holds up to
 * 64 requests beside the g / 16 GRU CTAs, larger batches run as consecutive launches inside the same call; the lock-step
 * kernel needs g / 16 + batch <= SM count and is simply not chosen otherwise. */
int dt_set_option(dt_handle *h, const char *name, int64_t value);

/* dt_get_option: read-back values; unknown name -> INVALID_ARG.  The device-side words synchronise the device first
 * (not capture-safe).
 *   "expand_path_taken"  expansion path the last dt_build_trees enqueued: 1 per-step kernels, 2 / 3 lock-step fused kernel
 *                        on mma.sync, 4 lock-step fused kernel on tcgen05, 5 wavefront kernel (dt_wave.cuh), 6 adaptive
 *                        (both persistent kernels enqueued, the device lets one run);
 *   "lockstep_speculation_used"  1 if the last lock-step launch speculated
 *   "schedule_chosen"    adaptive rounds: 1 if the last round's statistic said `flat` (wavefront kernel), else 0;
 *   "select_span_ns"     with "select_span" 1: device-side span of the last bulk select kernel (first CTA start to last
 *                        CTA end, %globaltimer);
 *   "state_slots"        GRU state slots per request in the workspace;
 *   "device_error"       1 after a hand-over wait inside a persistent kernel timed out (the round's outputs are invalid);
 *   "wave_steps", "wave_expansions"   dependent steps and CHILDREN evaluations request 0 needed in the last wavefront round. */
int dt_get_option(dt_handle *h, const char *name, int64_t *value);

/*
 * Phase timing (measurement aid, off by default).  dt_phase_timing(h, n_slots) creates n_slots
 * sets of CUDA events (n_slots = 0 frees them; not capture-safe).  While enabled, every
 * dt_build_trees call records the boundaries of its phases on `stream` into the slot chosen by
 * dt_phase_slot -- inside a stream capture as external event-record nodes, so each replay of the
 * captured graph re-records them.  dt_phase_elapsed_ms returns the device time of one phase of
 * the last completed round that used `slot` (the caller synchronises first); phases:
 *   DT_PHASE_SELECT (a1), DT_PHASE_PRECOMPUTE (a3, a4), DT_PHASE_EXPAND (a5-a8), DT_PHASE_EMIT (a9).
 */
#define DT_PHASE_SELECT 0
#define DT_PHASE_PRECOMPUTE 1
#define DT_PHASE_EXPAND 2
#define DT_PHASE_EMIT 3
#define DT_NUM_PHASES 4
int dt_phase_timing(dt_handle *h, int32_t n_slots);
int dt_phase_slot(dt_handle *h, int32_t slot);
int dt_phase_elapsed_ms(dt_handle *h, int32_t slot, int32_t phase, float *ms);

/* dt_kernel_launches: number of kernels the last dt_build_trees / dt_select_topm call enqueued. */
int64_t dt_kernel_launches(const dt_handle *h);

int dt_destroy(dt_handle *h);                 /* frees the workspace; h may be NULL           */
const char *dt_error_string(int code);        /* static string                                */
int dt_version(void);                         /* ABI version, currently 1                     */
size_t dt_workspace_bytes(const dt_handle *h);/* device bytes owned by the handle (incl. P)   */
int dt_last_cuda_error(const dt_handle *h);   /* cudaError_t of the last DT_ERR_CUDA          */

#ifdef __cplusplus
}
#endif
#endif /* DOMINOTREE_H */

// dt_api.cu -- host side of the C-ABI in include/dominotree.h: handle, validation, workspace,
// kernel launches.  Every launch goes to the caller's stream; dt_build_trees and dt_select_topm
// neither allocate nor synchronise, so a round can be captured into one CUDA graph.
#include <cuda_runtime.h>
#include <math.h>
#include <new>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>
#include <mutex>
#include <vector>

#include "../../include/dominotree.h"
#include "dt_budget.cuh"
#include "dt_commit.cuh"
#include "dt_expand.cuh"
#include "dt_frontier.cuh"
#include "dt_fused.cuh"
#include "dt_gemm_tc.cuh"
#include "dt_precompute.cuh"
#include "dt_scorers.cuh"
#include "dt_select.cuh"
#include "dt_wave.cuh"

using namespace dt;

struct dt_handle {
    dt_weights w;
    int max_batch, L, max_M, max_B, k;
    int heap_cap;
    size_t esize;
    // device workspace
    float *P;                       // [V, 3g]
    char *ws;                       // everything else, carved below
    size_t ws_bytes, p_bytes;
    int32_t *cand_id; float *cand_val;
    unsigned long long *sel_part; unsigned int *sel_counter, *sel_tau;
    float *C, *states, *heap_g; unsigned long long *heap_tp; int32_t *heap_cnt;
    // tensor-core precompute GEMM (bf16): split-K partials + tile tickets; side stream + fork/join events so the
    // GEMM overlaps the HBM-bound select inside the same round (and the same captured graph)
    float *mma_partial; unsigned int *mma_tickets; int mma_ok;
    float *tcg_partial; int tcg_ok;     // tcgen05 precompute GEMM: [kTcgSplits, rows_pad, r] partials
    cudaStream_t side; cudaEvent_t ev_fork, ev_join;
    // fused persistent expansion (bf16): state copies, split-K partials, hand-over words
    __nv_bfloat16 *s_hi, *s_lo; float *partial; unsigned long long *desc; unsigned int *flags, *round_ctr;
    int fused_ok, max_smem_optin;
    // wavefront expansion (dt_wave.cuh): per-item partials, multi-item descriptors, device error word, counters
    float *wv_partial; unsigned long long *wv_desc; unsigned int *wv_err, *wv_stats, *wv_flags, *wv_round; int wave_ok, slot_stride;
    int64_t opt_wave_width;         // items per request per step (0 = auto)
    int64_t opt_wave_groups;        // request groups the GRU CTAs serve in turn: 0 auto (2), 1 .. 4
    int64_t opt_adaptive;           // 1 (default): the device picks wavefront or lock-step per round (wave_regime_kernel)
    unsigned int *sched_sel;        // device word: sum over the rows of p1 in 16-bit fixed point (wave_regime_kernel)
    unsigned int sched_thr;         // wavefront schedule when the sum is below this
    int wave_clusters;              // co-resident clusters of kWvCS CTAs (0 = not queried yet, -1 = unavailable)
    int path_taken;                 // expansion path of the last dt_build_trees: 1 per-step, 2/3 fused mma.sync, 4 fused tcgen05, 5 wavefront,
                                    // 6 adaptive (wavefront or fused tcgen05 / mma.sync, chosen on the device per round)
    int64_t opt_expand_path;        // 0 auto, 1 per-step kernels, 2 fused mma.sync upc=8, 3 fused mma.sync upc=16, 4 fused tcgen05
    // host-call staging (lazy)
    char *stage; size_t stage_bytes;
    // options / bookkeeping
    int64_t opt_sel_span;           // 1: the bulk select kernel records its device-side span (first CTA start .. last CTA end)
    unsigned long long *sel_span;
    int64_t opt_fused_spec;         // lock-step kernel: speculative GRU pass along the chain (dt_fused.cuh)
    int64_t spec_used;              // the last lock-step launch speculated
    int64_t opt_fused_gsz;          // lock-step kernel: requests per group (0 = automatic)
    int64_t opt_gemm_serial;        // 1: the precompute GEMM runs after the select on the caller's stream (no overlap)
    int64_t opt_select_chunks;
    int64_t opt_select_kernel;      // 0 auto, 1 register-tile kernel only
    int64_t opt_schedule;           // 0 best-first heap (Alg. 1), 1 depth-synchronous frontier builder
    float *fr_state; int32_t *led_tok, *led_par, *led_cnt, *led_slot, *fr_ref, *fr_plane, *fr_n; float *led_g;
    int64_t opt_gemm;               // 0 auto (tcgen05 when the shape allows), 1 legacy mma.sync kernel
    int64_t opt_scorer;             // 0 DominoTree (Alg. 1), 1 Marg, 2 Cond-static
    int32_t *menu_tok; float *menu_lp;
    int sel_bulk_ok;
    // phase timing (optional): n_slots x kPhaseEvents events, recorded on the caller's stream
    cudaEvent_t *ph_ev; int ph_slots, ph_slot;
    int64_t launches;
    int last_cuda;
    int num_sms;
};

// The input-half table P = E W_ih^T (1.87 GB at the 8B shape) depends on the weights alone: handles created on the same
// borrowed weight tensors (same device, pointers, shapes, dtype -- e.g. one handle per stream of a serving process) share
// one copy, reference-counted; the weights are immutable while a handle borrows them (dominotree.h).
struct PEntry { const void *embed, *w_ih; int V, d, g, dtype, dev; float *P; int refs; };
static std::mutex g_p_mutex;
static std::vector<PEntry> g_p_cache;
static float *p_cache_acquire(const dt_weights &w, int dev) {
    std::lock_guard<std::mutex> lk(g_p_mutex);
    for (auto &e : g_p_cache)
        if (e.embed == w.embed && e.w_ih == w.gru_w_ih && e.V == w.V && e.d == w.d && e.g == w.g && e.dtype == (int)w.dtype && e.dev == dev) {
            e.refs += 1;
            return e.P;
        }
    return nullptr;
}
static void p_cache_insert(const dt_weights &w, int dev, float *P) {
    std::lock_guard<std::mutex> lk(g_p_mutex);
    g_p_cache.push_back(PEntry{w.embed, w.gru_w_ih, w.V, w.d, w.g, (int)w.dtype, dev, P, 1});
}
static void p_cache_release(float *P) {      // frees P when the last handle lets go (also for tables that never got into the cache)
    if (!P) return;
    std::lock_guard<std::mutex> lk(g_p_mutex);
    for (size_t i = 0; i < g_p_cache.size(); ++i)
        if (g_p_cache[i].P == P) {
            if (--g_p_cache[i].refs == 0) { cudaFree(P); g_p_cache.erase(g_p_cache.begin() + i); }
            return;
        }
    cudaFree(P);
}

#define DT_CUDA(h, call)                                                   \
    do {                                                                   \
        cudaError_t e__ = (call);                                          \
        if (e__ != cudaSuccess) { if (h) (h)->last_cuda = (int)e__; return DT_ERR_CUDA; } \
    } while (0)

static inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

// Phase boundaries of one round: [0] start, [1] after select (a1), [2] after precompute (a3, a4),
// [3] after the expansion loop (a5-a8), [4] after the emitter (a9).
constexpr int kPhaseEvents = DT_NUM_PHASES + 1;

// Record boundary `i` of the selected slot.  Inside a stream capture the record becomes an external
// event-record node, so every replay of the graph re-records it.
static int phase_mark(dt_handle *h, int i, cudaStream_t st) {
    if (!h->ph_ev) return DT_OK;
    cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
    DT_CUDA(h, cudaStreamIsCapturing(st, &cs));
    cudaEvent_t ev = h->ph_ev[(size_t)h->ph_slot * kPhaseEvents + i];
    DT_CUDA(h, cudaEventRecordWithFlags(ev, st, cs == cudaStreamCaptureStatusActive ? cudaEventRecordExternal
                                                                                   : cudaEventRecordDefault));
    return DT_OK;
}

extern "C" int dt_phase_timing(dt_handle *h, int32_t n_slots) {
    if (!h || n_slots < 0 || n_slots > 4096) return DT_ERR_INVALID_ARG;
    if (h->ph_ev) {
        for (int i = 0; i < h->ph_slots * kPhaseEvents; ++i) cudaEventDestroy(h->ph_ev[i]);
        free(h->ph_ev); h->ph_ev = nullptr; h->ph_slots = 0; h->ph_slot = 0;
    }
    if (n_slots == 0) return DT_OK;
    h->ph_ev = (cudaEvent_t *)calloc((size_t)n_slots * kPhaseEvents, sizeof(cudaEvent_t));
    if (!h->ph_ev) return DT_ERR_ALLOC;
    for (int i = 0; i < n_slots * kPhaseEvents; ++i) DT_CUDA(h, cudaEventCreate(&h->ph_ev[i]));
    h->ph_slots = n_slots;
    return DT_OK;
}
extern "C" int dt_phase_slot(dt_handle *h, int32_t slot) {
    if (!h || !h->ph_ev || slot < 0 || slot >= h->ph_slots) return DT_ERR_INVALID_ARG;
    h->ph_slot = slot;
    return DT_OK;
}
extern "C" int dt_phase_elapsed_ms(dt_handle *h, int32_t slot, int32_t phase, float *ms) {
    if (!h || !h->ph_ev || !ms || slot < 0 || slot >= h->ph_slots || phase < 0 || phase >= DT_NUM_PHASES)
        return DT_ERR_INVALID_ARG;
    const cudaEvent_t *e = h->ph_ev + (size_t)slot * kPhaseEvents;
    DT_CUDA(h, cudaEventElapsedTime(ms, e[phase], e[phase + 1]));
    return DT_OK;
}

extern "C" const char *dt_error_string(int code) {
    switch (code) {
        case DT_OK: return "ok";
        case DT_ERR_INVALID_ARG: return "invalid argument";
        case DT_ERR_UNSUPPORTED: return "unsupported shape (beyond compiled limits)";
        case DT_ERR_CUDA: return "CUDA runtime error";
        case DT_ERR_ALLOC: return "allocation failed";
        case DT_ERR_STATIC_LIMIT: return "shape beyond the static scratch limits (DT_STATIC_MAX_ROWS rows, DT_MAX_M candidates)";
        default: return "unknown error";
    }
}
extern "C" int dt_version(void) { return 1; }
extern "C" size_t dt_workspace_bytes(const dt_handle *h) { return h ? h->ws_bytes + h->p_bytes + h->stage_bytes : 0; }
extern "C" int dt_last_cuda_error(const dt_handle *h) { return h ? h->last_cuda : 0; }
extern "C" int64_t dt_kernel_launches(const dt_handle *h) { return h ? h->launches : 0; }

extern "C" int dt_set_option(dt_handle *h, const char *name, int64_t value) {
    if (!h || !name) return DT_ERR_INVALID_ARG;
    if (!strcmp(name, "wave_width")) {
        if (value < 0 || value > kWvMaxW) return DT_ERR_INVALID_ARG;
        h->opt_wave_width = value;
        return DT_OK;
    }
    if (!strcmp(name, "wave_groups")) {
        if (value < 0 || value > 4) return DT_ERR_INVALID_ARG;
        h->opt_wave_groups = value;
        return DT_OK;
    }
    if (!strcmp(name, "adaptive_schedule")) {
        if (value < 0 || value > 1) return DT_ERR_INVALID_ARG;
        h->opt_adaptive = value;
        return DT_OK;
    }
    if (!strcmp(name, "expand_path")) {
        if (value < 0 || value > 5) return DT_ERR_INVALID_ARG;
        h->opt_expand_path = value;
        return DT_OK;
    }
    if (!strcmp(name, "schedule")) {
        if (value < 0 || value > 1) return DT_ERR_INVALID_ARG;
        h->opt_schedule = value;
        return DT_OK;
    }
    if (!strcmp(name, "precompute_gemm")) {
        if (value < 0 || value > 1) return DT_ERR_INVALID_ARG;
        h->opt_gemm = value;
        return DT_OK;
    }
    if (!strcmp(name, "scorer")) {
        if (value < 0 || value > 2) return DT_ERR_INVALID_ARG;
        h->opt_scorer = value;
        return DT_OK;
    }
    if (!strcmp(name, "select_span")) { h->opt_sel_span = value; return DT_OK; }
    if (!strcmp(name, "precompute_serial")) { h->opt_gemm_serial = value; return DT_OK; }
    if (!strcmp(name, "lockstep_speculation")) { if (value < 0 || value > 2) return DT_ERR_INVALID_ARG; h->opt_fused_spec = value; return DT_OK; }
    if (!strcmp(name, "lockstep_group")) { if (value < 0 || value > kFusChunk) return DT_ERR_INVALID_ARG; h->opt_fused_gsz = value; return DT_OK; }
    if (!strcmp(name, "select_kernel")) {
        if (value < 0 || value > 1) return DT_ERR_INVALID_ARG;
        h->opt_select_kernel = value;
        return DT_OK;
    }
    if (!strcmp(name, "select_chunks")) {
        if (value < 0 || value > kSelMaxChunks) return DT_ERR_INVALID_ARG;
        h->opt_select_chunks = value;
        return DT_OK;
    }
    return DT_ERR_INVALID_ARG;
}

// Read-back knobs (synchronise the device for the device-side words; not capture-safe).
extern "C" int dt_get_option(dt_handle *h, const char *name, int64_t *value) {
    if (!h || !name || !value) return DT_ERR_INVALID_ARG;
    if (!strcmp(name, "expand_path_taken")) { *value = h->path_taken; return DT_OK; }
    if (!strcmp(name, "state_slots")) { *value = h->slot_stride; return DT_OK; }
    if (!strcmp(name, "lockstep_speculation_used")) { *value = h->spec_used; return DT_OK; }
    const bool dev_word = !strcmp(name, "device_error") || !strcmp(name, "wave_steps") || !strcmp(name, "wave_expansions") ||
                          !strcmp(name, "schedule_chosen") || !strcmp(name, "select_span_ns");
    if (!dev_word) return DT_ERR_INVALID_ARG;
    *value = 0;
    if (!h->wv_err) return DT_OK;
    unsigned int w[40];
    DT_CUDA(h, cudaDeviceSynchronize());
    DT_CUDA(h, cudaMemcpy(w, h->wv_err, sizeof(w), cudaMemcpyDeviceToHost));
    if (!strcmp(name, "select_span_ns")) {
        const unsigned long long t0 = ((unsigned long long)w[33] << 32) | w[32], t1 = ((unsigned long long)w[35] << 32) | w[34];
        *value = (t1 > t0) ? (int64_t)(t1 - t0) : 0;
        return DT_OK;
    }
    *value = !strcmp(name, "device_error") ? w[0] : !strcmp(name, "wave_steps") ? w[8] : !strcmp(name, "wave_expansions") ? w[9] : (w[16] < h->sched_thr ? 1 : 0);
    return DT_OK;
}

template <typename T>
static int launch_gemm_nt(dt_handle *h, const void *A, long long lda, const void *Bm, long long ldb,
                          float *out, long long ldo, int Mr, int Nc, int K, cudaStream_t st) {
    dim3 grid((Nc + kGemmBN - 1) / kGemmBN, (Mr + kGemmBM - 1) / kGemmBM);
    gemm_nt_kernel<T><<<grid, 256, 0, st>>>(reinterpret_cast<const T *>(A), lda, reinterpret_cast<const T *>(Bm), ldb,
                                            out, ldo, Mr, Nc, K);
    h->launches++;
    DT_CUDA(h, cudaGetLastError());
    return DT_OK;
}

// C = H W1[:, 0:d]^T on the tensor cores (dt_gemm_mma.cuh), split-K kMmaSplits ways.
constexpr int kMmaSplits = 16;
static int launch_gemm_mma(dt_handle *h, const void *A, long long lda, const void *Bm, long long ldb,
                           float *out, long long ldo, int Mr, int Nc, int K, cudaStream_t st) {
    GemmMmaParams g;
    g.A = reinterpret_cast<const __nv_bfloat16 *>(A); g.lda = lda;
    g.Bm = reinterpret_cast<const __nv_bfloat16 *>(Bm); g.ldb = ldb;
    g.out = out; g.ldo = ldo; g.M = Mr; g.N = Nc; g.K = K;
    const int tm = (Mr + kMmaBM - 1) / kMmaBM, tn = (Nc + kMmaBN - 1) / kMmaBN;
    // The K split depends on K only, never on the batch: every output element is then summed in the same order
    // whatever the batch size (batch invariance).
    const int kt = (K + kMmaBK - 1) / kMmaBK;
    int splits = kt < kMmaSplits ? kt : kMmaSplits;
    g.k_per_split = ((kt + splits - 1) / splits) * kMmaBK;
    splits = (K + g.k_per_split - 1) / g.k_per_split;
    g.splits = splits; g.partial = h->mma_partial; g.tile_counter = h->mma_tickets;
    dim3 grid(tn, tm, splits);
    gemm_nt_bf16_mma_kernel<<<grid, kMmaThreads, 0, st>>>(g);
    h->launches++;
    DT_CUDA(h, cudaGetLastError());
    return DT_OK;
}

// C = H W1[:, 0:d]^T on tcgen05 (dt_gemm_tc.cuh): split-K partials, then the fixed-order reduction.
static int launch_gemm_tc(dt_handle *h, const void *A, long long lda, const void *Bm, long long ldb,
                          float *out, long long ldo, int Mr, int Nc, int K, cudaStream_t st) {
    GemmTcParams g;
    g.A = reinterpret_cast<const __nv_bfloat16 *>(A); g.lda = lda;
    g.Bm = reinterpret_cast<const __nv_bfloat16 *>(Bm); g.ldb = ldb;
    g.partial = h->tcg_partial; g.out = out; g.ldo = ldo;
    g.Mr = Mr; g.Nc = Nc; g.K = K; g.Mr_pad = (Mr + 127) / 128 * 128;
    gemm_c_tc_kernel<<<dim3(g.Mr_pad / 128, kTcgSplits), kTcgThreads, gemm_tc_smem(), st>>>(g);
    const long long n = (long long)Mr * (Nc / 4);
    gemm_c_reduce_kernel<<<(unsigned int)((n + 255) / 256), 256, 0, st>>>(g);
    h->launches += 2;
    DT_CUDA(h, cudaGetLastError());
    return DT_OK;
}

extern "C" int dt_create(dt_handle **out, const dt_weights *w, int32_t max_batch, int32_t L,
                         int32_t max_M, int32_t max_B, int32_t k) {
    if (!out || !w) return DT_ERR_INVALID_ARG;
    *out = nullptr;
    if (!w->embed || !w->gru_w_ih || !w->gru_w_hh || !w->corr_w1 || !w->corr_w2) return DT_ERR_INVALID_ARG;
    if (w->V < 1 || w->d < 1 || w->g < 1 || w->r < 1) return DT_ERR_INVALID_ARG;
    if (w->dtype != DT_BF16 && w->dtype != DT_F32) return DT_ERR_INVALID_ARG;
    if (max_batch < 1 || L < 1 || max_B < 1 || k < 1 || max_M < k || max_M > w->V) return DT_ERR_INVALID_ARG;
    if (max_M > DT_MAX_M || max_B > DT_MAX_B || k > DT_MAX_K || L > DT_MAX_L) return DT_ERR_UNSUPPORTED;

    dt_handle *h = new (std::nothrow) dt_handle();
    if (!h) return DT_ERR_ALLOC;
    memset(h, 0, sizeof(*h));
    h->w = *w;
    h->max_batch = max_batch; h->L = L; h->max_M = max_M; h->max_B = max_B; h->k = k;
    h->heap_cap = max_B * k + k;
    h->opt_adaptive = 1;
    h->opt_fused_spec = 1;
    h->esize = (w->dtype == DT_BF16) ? 2 : 4;
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess ||
        cudaDeviceGetAttribute(&h->num_sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) {
        delete h; return DT_ERR_CUDA;
    }

    const size_t rows = (size_t)max_batch * L;
    size_t off = 0;
    auto carve = [&](size_t bytes) { size_t o = off; off = align_up(off + bytes, 256); return o; };
    const size_t o_cid = carve(rows * max_M * 4), o_cval = carve(rows * max_M * 4);
    const size_t o_part = carve(rows * kSelMaxChunks * (size_t)max_M * 8);
    const size_t o_cnt = carve(rows * 4), o_tau = carve(rows * 4);
    const size_t o_C = carve(rows * w->r * 4);
    // state slots per request: slot 0 = zeros, expansion x at x + 1; the wavefront schedule may expand up to 2 max_B + 1
    // nodes (speculative picks included), static mode walks L nodes
    const size_t slots = (size_t)((2 * max_B > L) ? 2 * max_B : L) + 2;
    h->slot_stride = (int)slots;
    const size_t o_states = carve((size_t)max_batch * slots * w->g * 4);
    // fused path eligibility (shape part; the grid / smem fit is checked per call)
    h->fused_ok = (w->dtype == DT_BF16) && (w->g % 32 == 0) && (w->r % 8 == 0) && max_M <= 256 &&
                  ((reinterpret_cast<uintptr_t>(w->gru_w_hh) & 15u) == 0) && ((reinterpret_cast<uintptr_t>(w->corr_w2) & 15u) == 0);
    size_t o_shi = 0, o_slo = 0, o_partial = 0, o_desc = 0, o_sync = 0, o_wpart = 0, o_wdesc = 0, o_werr = 0, o_wsync = 0;
    if (h->fused_ok) {
        o_shi = carve((size_t)max_batch * slots * w->g * 2);
        o_slo = carve((size_t)max_batch * slots * w->g * 2);
        o_partial = carve((size_t)(w->g / 8) * max_batch * w->r * 4);
        o_desc = carve((size_t)max_batch * 8 * kFusDescStride);
        o_sync = carve((size_t)256 * 4 * kFusFlagStride + 256);
        o_wpart = carve((size_t)max_batch * kWvMaxW * (w->g / 16 + 1) * w->r * 4);
        o_wdesc = carve((size_t)max_batch * kWvDescWords * 8);
        o_werr = carve(256);
        o_wsync = carve((size_t)256 * 4 * kFusFlagStride + 256);   // the wavefront kernel's own flags + round counter (its tags differ)
    }
    // MMA GEMM eligibility: bf16, 16-byte aligned rows of H and W1
    h->mma_ok = (w->dtype == DT_BF16) && (w->d % 8 == 0) && ((w->d + w->g) % 8 == 0) &&
                ((reinterpret_cast<uintptr_t>(w->corr_w1) & 15u) == 0);
    const size_t mma_tiles = ((rows + kMmaBM - 1) / kMmaBM) * (size_t)((w->r + kMmaBN - 1) / kMmaBN);
    size_t o_mpart = 0, o_mtick = 0;
    if (h->mma_ok) {
        o_mpart = carve(mma_tiles * kMmaSplits * (size_t)kMmaBM * kMmaBN * 4);
        o_mtick = carve(mma_tiles * 4);
    }
    const size_t o_mtok = carve(rows * k * 4), o_mlp = carve(rows * k * 4);
    const size_t rows_pad = (rows + 127) / 128 * 128;
    h->tcg_ok = h->mma_ok && (w->d % (64 * kTcgSplits) == 0) && (w->r % 16 == 0) && w->r <= 256 && h->opt_gemm != 1;
    const size_t o_tcg = h->tcg_ok ? carve((size_t)kTcgSplits * rows_pad * w->r * 4) : 0;
    // frontier schedule: lane states (ping-pong), ledger, frontier lists
    const size_t led_n = (size_t)max_batch * L * max_B * k;
    const size_t o_fst = carve((size_t)2 * max_batch * max_B * w->g * 4);
    const size_t o_ltok = carve(led_n * 4), o_lpar = carve(led_n * 4), o_lg = carve(led_n * 4), o_lslot = carve(led_n * 4);
    const size_t o_lcnt = carve(rows * 4), o_fref = carve((size_t)2 * max_batch * max_B * 4), o_fpl = carve((size_t)2 * max_batch * max_B * 4);
    const size_t o_fn = carve((size_t)2 * max_batch * 4);
    const size_t o_hg = carve((size_t)max_batch * h->heap_cap * 4);
    const size_t o_htp = carve((size_t)max_batch * h->heap_cap * 8);
    const size_t o_hcnt = carve((size_t)max_batch * 4);
    h->ws_bytes = off;
    h->p_bytes = (size_t)w->V * 3 * w->g * 4;
    if (cudaMalloc(&h->ws, h->ws_bytes) != cudaSuccess) { cudaGetLastError(); delete h; return DT_ERR_ALLOC; }
    bool p_shared = false;
    h->P = p_cache_acquire(*w, dev);
    if (h->P) p_shared = true;
    else if (cudaMalloc(&h->P, h->p_bytes) != cudaSuccess) { cudaGetLastError(); cudaFree(h->ws); delete h; return DT_ERR_ALLOC; }
    h->cand_id = (int32_t *)(h->ws + o_cid); h->cand_val = (float *)(h->ws + o_cval);
    h->sel_part = (unsigned long long *)(h->ws + o_part);
    h->sel_counter = (unsigned int *)(h->ws + o_cnt); h->sel_tau = (unsigned int *)(h->ws + o_tau);
    h->C = (float *)(h->ws + o_C); h->states = (float *)(h->ws + o_states);
    h->heap_g = (float *)(h->ws + o_hg); h->heap_tp = (unsigned long long *)(h->ws + o_htp);
    h->heap_cnt = (int32_t *)(h->ws + o_hcnt);
    h->menu_tok = (int32_t *)(h->ws + o_mtok); h->menu_lp = (float *)(h->ws + o_mlp);
    h->fr_state = (float *)(h->ws + o_fst); h->led_tok = (int32_t *)(h->ws + o_ltok); h->led_par = (int32_t *)(h->ws + o_lpar);
    h->led_g = (float *)(h->ws + o_lg); h->led_slot = (int32_t *)(h->ws + o_lslot); h->led_cnt = (int32_t *)(h->ws + o_lcnt);
    h->fr_ref = (int32_t *)(h->ws + o_fref); h->fr_plane = (int32_t *)(h->ws + o_fpl); h->fr_n = (int32_t *)(h->ws + o_fn);
    if (h->tcg_ok) {
        h->tcg_partial = (float *)(h->ws + o_tcg);
        if (cudaFuncSetAttribute(gemm_c_tc_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)gemm_tc_smem()) != cudaSuccess) { cudaGetLastError(); h->tcg_ok = 0; }
    }
    if (h->mma_ok) { h->mma_partial = (float *)(h->ws + o_mpart); h->mma_tickets = (unsigned int *)(h->ws + o_mtick); }
    if (cudaStreamCreateWithFlags(&h->side, cudaStreamNonBlocking) != cudaSuccess ||
        cudaEventCreateWithFlags(&h->ev_fork, cudaEventDisableTiming) != cudaSuccess ||
        cudaEventCreateWithFlags(&h->ev_join, cudaEventDisableTiming) != cudaSuccess) {
        cudaGetLastError(); cudaFree(h->ws); p_cache_release(h->P); delete h; return DT_ERR_CUDA;
    }
    if (h->fused_ok) {
        h->s_hi = (__nv_bfloat16 *)(h->ws + o_shi); h->s_lo = (__nv_bfloat16 *)(h->ws + o_slo);
        h->partial = (float *)(h->ws + o_partial); h->desc = (unsigned long long *)(h->ws + o_desc);
        h->flags = (unsigned int *)(h->ws + o_sync);
        h->round_ctr = h->flags + (size_t)256 * kFusFlagStride;
        h->wv_partial = (float *)(h->ws + o_wpart); h->wv_desc = (unsigned long long *)(h->ws + o_wdesc);
        h->wv_err = (unsigned int *)(h->ws + o_werr); h->wv_stats = h->wv_err + 8; h->sched_sel = h->wv_err + 16; h->sel_span = reinterpret_cast<unsigned long long *>(h->wv_err + 32);
        h->wv_flags = (unsigned int *)(h->ws + o_wsync); h->wv_round = h->wv_flags + (size_t)256 * kFusFlagStride;
        h->wave_ok = (slots <= 1023);
        bool ok = cudaDeviceGetAttribute(&h->max_smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev) == cudaSuccess;
        h->max_smem_optin -= 1024;                  // room for the kernels' static shared memory
        if (!ok ||
            cudaFuncSetAttribute(fused_expand_kernel<8>, cudaFuncAttributeMaxDynamicSharedMemorySize, h->max_smem_optin) != cudaSuccess ||
            cudaFuncSetAttribute(fused_expand_kernel<16>, cudaFuncAttributeMaxDynamicSharedMemorySize, h->max_smem_optin) != cudaSuccess ||
            cudaFuncSetAttribute(fused_expand_kernel<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, h->max_smem_optin) != cudaSuccess) {
            cudaGetLastError(); h->fused_ok = 0; h->wave_ok = 0;
        }
        if (h->wave_ok && cudaFuncSetAttribute(wave_expand_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, h->max_smem_optin) != cudaSuccess) {
            cudaGetLastError(); h->wave_ok = 0;
        }
    }

    h->sel_bulk_ok =
        cudaFuncSetAttribute(select_topm_bulk_kernel<__nv_bfloat16, SelectSmemBig>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sel_bulk_dyn_smem<SelectSmemBig>()) == cudaSuccess &&
        cudaFuncSetAttribute(select_topm_bulk_kernel<float, SelectSmemBig>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sel_bulk_dyn_smem<SelectSmemBig>()) == cudaSuccess &&
        cudaFuncSetAttribute(select_topm_bulk_kernel<__nv_bfloat16, SelectSmemW4>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sel_bulk_dyn_smem<SelectSmemW4>()) == cudaSuccess &&
        cudaFuncSetAttribute(select_topm_bulk_kernel<float, SelectSmemW4>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sel_bulk_dyn_smem<SelectSmemW4>()) == cudaSuccess;
    if (!h->sel_bulk_ok) cudaGetLastError();
    int rc = DT_OK;
    if (cudaMemset(h->ws, 0, h->ws_bytes) != cudaSuccess) rc = DT_ERR_CUDA;
    {   // dynamic shared memory of expand_kernel at the handle's maxima
        const size_t dsm = (size_t)(w->g + w->r + max_M) * 4 + (size_t)max_M * 4;
        if (dsm > 200 * 1024) rc = DT_ERR_UNSUPPORTED;
        else if (dsm > 48 * 1024) {
            cudaError_t e = (w->dtype == DT_BF16)
                ? cudaFuncSetAttribute(expand_kernel<__nv_bfloat16>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)dsm)
                : cudaFuncSetAttribute(expand_kernel<float>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)dsm);
            if (e != cudaSuccess) rc = DT_ERR_CUDA;
        }
    }
    // P = E W_ih^T  (weight-only table)
    if (rc == DT_OK && !p_shared) {
        if (w->dtype == DT_BF16)
            rc = launch_gemm_nt<__nv_bfloat16>(h, w->embed, w->d, w->gru_w_ih, w->d, h->P, 3LL * w->g, w->V, 3 * w->g, w->d, 0);
        else
            rc = launch_gemm_nt<float>(h, w->embed, w->d, w->gru_w_ih, w->d, h->P, 3LL * w->g, w->V, 3 * w->g, w->d, 0);
    }
    if (rc == DT_OK && cudaDeviceSynchronize() != cudaSuccess) { h->last_cuda = (int)cudaGetLastError(); rc = DT_ERR_CUDA; }
    if (rc != DT_OK) { cudaFree(h->ws); p_cache_release(h->P); delete h; return rc; }
    if (!p_shared) p_cache_insert(*w, dev, h->P);
    h->launches = 0;
    *out = h;
    return DT_OK;
}

extern "C" int dt_destroy(dt_handle *h) {
    if (!h) return DT_OK;
    dt_phase_timing(h, 0);
    if (h->side) cudaStreamDestroy(h->side);
    if (h->ev_fork) cudaEventDestroy(h->ev_fork);
    if (h->ev_join) cudaEventDestroy(h->ev_join);
    cudaFree(h->ws); p_cache_release(h->P);
    if (h->stage) cudaFree(h->stage);
    delete h;
    return DT_OK;
}

static int pick_chunks(const dt_handle *h, int rows, int M, int cap, int row_vecs) {
    int smax = cap / M;                             // the merging CTA holds S * M keys in its candidate buffer
    if (smax > kSelMaxChunks) smax = kSelMaxChunks;
    if (smax < 1) smax = 1;
    int S;
    if (h->opt_select_chunks > 0) S = (int)h->opt_select_chunks;
    else {
        const int target = 3 * h->num_sms;          // resident CTAs wanted
        S = (target + rows - 1) / rows;
        // A chunk must keep all 8 warps of its CTA busy for a few tiles, or their threshold claims are worthless
        // and everything is pushed (measured at batch 1, V = 151 936: S = 4 -> 16 us, S = 28 -> 390 us).
        int by_len = row_vecs / 4096;
        if (by_len < 1) by_len = 1;
        if (S > by_len) S = by_len;
    }
    if (S > smax) S = smax;
    if (S < 1) S = 1;
    return S;
}

static int launch_select(dt_handle *h, const void *logits, int rows, int M, int32_t *cand_id, float *cand_val,
                         cudaStream_t st) {
    const int V = h->w.V;
    const int kvec = (h->w.dtype == DT_BF16) ? 8 : 4;
    const bool aligned = (V % kvec == 0) && ((reinterpret_cast<uintptr_t>(logits) & 15u) == 0);
    // bulk-copy kernel (cp.async.bulk ring per warp) for 16-byte aligned rows, else the register-tile kernel
    const bool bulk = aligned && h->opt_select_kernel != 1 && h->sel_bulk_ok;
    SelectParams p;
    p.logits = logits; p.rows = rows; p.V = V; p.M = M;
    p.row_vecs = (V + kvec - 1) / kvec;
    const bool w4 = false;                       // (4-warp CTAs, four per SM: measured slower, looser threshold claims)
    int S = pick_chunks(h, rows, M, w4 ? SelectSmemW4::kCap : SelectSmemBig::kCap, p.row_vecs);
    if (S > p.row_vecs) S = p.row_vecs;
    p.S = S;
    p.chunk_vecs = (p.row_vecs + S - 1) / S;
    if (bulk) p.chunk_vecs = (p.chunk_vecs + kSelTileVecs - 1) / kSelTileVecs * kSelTileVecs;   // chunks start on tile boundaries
    p.cand_id = cand_id; p.cand_val = cand_val;
    p.part = h->sel_part; p.row_counter = h->sel_counter; p.row_tau = h->sel_tau;
    p.span = nullptr;
    if (h->opt_sel_span && bulk && h->sel_span) {
        p.span = h->sel_span;
        DT_CUDA(h, cudaMemsetAsync(h->sel_span, 0xFF, 8, st));
        DT_CUDA(h, cudaMemsetAsync(h->sel_span + 1, 0, 8, st));
    }
    dim3 grid(S, rows);
    if (bulk) {
        if (h->w.dtype == DT_BF16) {
            if (w4) select_topm_bulk_kernel<__nv_bfloat16, SelectSmemW4><<<grid, 128, sel_bulk_dyn_smem<SelectSmemW4>(), st>>>(p);
            else select_topm_bulk_kernel<__nv_bfloat16, SelectSmemBig><<<grid, 256, sel_bulk_dyn_smem<SelectSmemBig>(), st>>>(p);
        } else {
            if (w4) select_topm_bulk_kernel<float, SelectSmemW4><<<grid, 128, sel_bulk_dyn_smem<SelectSmemW4>(), st>>>(p);
            else select_topm_bulk_kernel<float, SelectSmemBig><<<grid, 256, sel_bulk_dyn_smem<SelectSmemBig>(), st>>>(p);
        }
    } else if (h->w.dtype == DT_BF16) {
        if (aligned) select_topm_kernel<__nv_bfloat16, true><<<grid, kSelThreads, 0, st>>>(p);
        else select_topm_kernel<__nv_bfloat16, false><<<grid, kSelThreads, 0, st>>>(p);
    } else {
        if (aligned) select_topm_kernel<float, true><<<grid, kSelThreads, 0, st>>>(p);
        else select_topm_kernel<float, false><<<grid, kSelThreads, 0, st>>>(p);
    }
    h->launches++;
    DT_CUDA(h, cudaGetLastError());
    return DT_OK;
}

extern "C" int dt_select_topm(dt_handle *h, const void *logits, int32_t rows, int32_t M,
                              int32_t *cand_id, float *cand_val, void *stream) {
    if (!h) return DT_ERR_INVALID_ARG;
    if (rows < 0 || rows > h->max_batch * h->L || M < 1 || M > h->max_M) return DT_ERR_INVALID_ARG;
    h->launches = 0;
    if (rows == 0) return DT_OK;
    if (!logits || !cand_id || !cand_val) return DT_ERR_INVALID_ARG;
    return launch_select(h, logits, rows, M, cand_id, cand_val, (cudaStream_t)stream);
}

// Fused persistent expansion (dt_fused.cuh).  Returns 1 if the shape does not fit (caller falls back
// to the per-step kernels), DT_OK after enqueueing, or a negative error.
// `sel` >= 0: adaptive round, the kernel runs only when the device's schedule word equals it; `probe`: only report the fit;
// `m_begin` / `m_end`: record the phase marks in front of / behind the launch
static int launch_fused(dt_handle *h, ExpandParams &p, cudaStream_t st, bool static_mode = false, int sel = -1, bool probe = false,
                        bool m_begin = true, bool m_end = true) {
    if (!h->fused_ok || h->opt_expand_path == 1) return 1;
    // one-step rounds: GRU CTA 0 would bump the round counter before a late-starting CTA has read it
    if (p.B < 2) return 1;
    int upc = 0;
    bool tcgen = false;
    // tcgen05 + TMEM GRU CTAs (16 units each) whenever the shape allows; the choice never depends on the batch
    // beyond fitting on the chip, so results stay batch-invariant
    if ((h->opt_expand_path == 0 || h->opt_expand_path == 4) && p.g % kTcKC == 0 && p.r % 8 == 0 && p.r <= 256 &&
        p.g / kTcUPC + p.batch <= h->num_sms && p.g / kTcUPC <= 256 && (size_t)16 * p.g * 2 <= (size_t)kTcSlots * kTcSlotBytes &&
        fused_tc_smem(p.g, p.r) <= (size_t)h->max_smem_optin) {
        tcgen = true; upc = kTcUPC;
    }
    if (h->opt_expand_path == 4 && !tcgen) return 1;
    for (int cand : {16, 8}) {      // mma.sync fallback; batch-independent preference => batch-invariant results
        if (tcgen) break;
        if (h->opt_expand_path == 2 && cand != 8) continue;
        if (h->opt_expand_path == 3 && cand != 16) continue;
        if (p.g % cand) continue;
        if (p.g / cand + p.batch > h->num_sms || p.g / cand > 256) continue;
        const int mt = (3 * cand + 15) / 16;
        if (fused_gru_smem(p.g, p.r, cand, mt) > (size_t)h->max_smem_optin) continue;
        upc = cand; break;
    }
    if (!upc) return 1;
    FusedParams f;
    memset(&f, 0, sizeof(f));
    f.e = p;
    f.upc = upc; f.n_gru = p.g / upc; f.m_tiles = (3 * upc + 15) / 16;
    // two groups when the batch allows (ping-pong between the GRU CTAs and the request CTAs), at most kFusChunk requests each
    f.gsz = (p.batch <= 16) ? p.batch : ((p.batch + 1) / 2 < kFusChunk ? (p.batch + 1) / 2 : kFusChunk);
    // Speculation along the chain (dt_fused.cuh): by default on the rounds the adaptive schedule sends here, i.e. peaked
    // ones, where most pops are the marginal top-1 child of the node just expanded (a hit overlaps the GRU pass with the
    // request CTA's scoring, a miss costs a second pass); option 2 forces it, 0 disables it.  tcgen05 role only (its
    // n_gru = g / 16 leaves room for a second partial buffer in the workspace, sized for g / 8 CTAs); token ids must leave
    // the descriptor's top byte to the depth.  One group of up to 32 requests then: a hit's period is one pass.
    const bool want_spec = h->opt_fused_spec == 2 || (h->opt_fused_spec == 1 && !static_mode);
    f.spec = (tcgen && want_spec && p.V <= (1 << 24)) ? 1 : 0;
    if (f.spec) f.gsz = p.batch < kFusChunk ? p.batch : kFusChunk;
    if (h->opt_fused_gsz > 0) f.gsz = (int)h->opt_fused_gsz < p.batch ? (int)h->opt_fused_gsz : p.batch;
    // (several groups share the GRU CTAs: their passes queue up behind one another and the speculation only adds passes;
    // measured at batch 40: 491 vs 461 us per peaked round)
    if (f.spec && h->opt_fused_spec != 2 && p.batch > f.gsz) { f.spec = 0; f.gsz = (p.batch + 1) / 2 < kFusChunk ? (p.batch + 1) / 2 : kFusChunk; }
    if ((p.batch + f.gsz - 1) / f.gsz > kFusMaxGroups) f.spec = 0;
    f.partial_buf = (size_t)(p.g / 16) * h->max_batch * p.r;
    f.slot_stride = h->slot_stride;
    f.s_hi = h->s_hi; f.s_lo = h->s_lo; f.s32 = h->states; f.partial = h->partial; f.desc = h->desc; f.flags = h->flags; f.round_ctr = h->round_ctr;
    f.static_mode = static_mode ? 1 : 0; f.menu_tok = h->menu_tok; f.menu_lp = h->menu_lp; f.err = h->wv_err;
    f.w2_smem = 1; f.w2_bufs = 2;
    size_t rs = fused_req_smem(p.r, p.M, p.N, p.k, 1, 2);
    if (rs > (size_t)h->max_smem_optin) { f.w2_bufs = 1; rs = fused_req_smem(p.r, p.M, p.N, p.k, 1, 1); }
    if (rs > (size_t)h->max_smem_optin) { f.w2_smem = 0; rs = fused_req_smem(p.r, p.M, p.N, p.k, 0); }
    if (rs > (size_t)h->max_smem_optin) return 1;
    const size_t gs = tcgen ? fused_tc_smem(p.g, p.r) : fused_gru_smem(p.g, p.r, upc, f.m_tiles);
    const size_t dsm = gs > rs ? gs : rs;
    if (probe) return DT_OK;
    h->spec_used = f.spec;
    f.stats = h->wv_stats;                           // read back as "wave_steps" / "wave_expansions"
    if (sel >= 0) { f.sched_sel = h->sched_sel; f.sched_want = (unsigned int)sel; f.sched_thr = h->sched_thr; }
    int rc = m_begin ? phase_mark(h, 2, st) : DT_OK;
    if (rc) return rc;
    void *args[] = {&f};
    const dim3 grid(f.n_gru + p.batch), block(kFusThreads);
    cudaError_t e = tcgen ? cudaLaunchCooperativeKernel((const void *)fused_expand_kernel<0>, grid, block, args, dsm, st)
                  : (upc == 8) ? cudaLaunchCooperativeKernel((const void *)fused_expand_kernel<8>, grid, block, args, dsm, st)
                               : cudaLaunchCooperativeKernel((const void *)fused_expand_kernel<16>, grid, block, args, dsm, st);
    h->launches++;
    DT_CUDA(h, e);
    h->path_taken = tcgen ? 4 : (upc == 8 ? 2 : 3);
    if (static_mode || !m_end) return DT_OK;
    if ((rc = phase_mark(h, 3, st))) return rc;
    return phase_mark(h, 4, st);
}

// Wavefront expansion (dt_wave.cuh).  Returns 1 if the shape does not fit (caller falls back to the lock-step fused
// kernel), DT_OK after enqueueing, or a negative error.  Batches beyond what one cooperative launch holds (one request
// CTA per request beside the g / 16 GRU CTAs) are split into consecutive launches: no cliff, requests are independent.
static int launch_wave(dt_handle *h, ExpandParams &p, cudaStream_t st, int sel = -1, bool probe = false, bool m_begin = true,
                       bool m_end = true) {
    if (!h->fused_ok || !h->wave_ok || (h->opt_expand_path != 0 && h->opt_expand_path != 5)) return 1;
    if (p.g % kWvKC || p.g / 16 > 256 || p.r % 8 || p.r > 256 || p.k > 32 || p.M > 256 || p.L > DT_MAX_L || p.V > (1 << 20)) return 1;
    const int n_gru = p.g / 16;                          // a multiple of kWvCS (g is a multiple of 128)
    const size_t gs = wave_gru_smem(p.g, p.r);
    if (gs > (size_t)h->max_smem_optin) return 1;
    // co-resident clusters of kWvCS CTAs at one CTA per SM (queried once per handle)
    if (h->wave_clusters == 0) {
        cudaLaunchConfig_t qc;
        memset(&qc, 0, sizeof(qc));
        qc.gridDim = dim3(h->num_sms / kWvCS * kWvCS); qc.blockDim = dim3(kWvThreads); qc.dynamicSmemBytes = (size_t)h->max_smem_optin;
        cudaLaunchAttribute qa[1];
        qa[0].id = cudaLaunchAttributeClusterDimension; qa[0].val.clusterDim.x = kWvCS; qa[0].val.clusterDim.y = 1; qa[0].val.clusterDim.z = 1;
        qc.attrs = qa; qc.numAttrs = 1;
        int nc = 0;
        if (cudaOccupancyMaxActiveClusters(&nc, (const void *)wave_expand_kernel, &qc) != cudaSuccess) { cudaGetLastError(); nc = -1; }
        h->wave_clusters = nc > 0 ? nc : -1;
    }
    if (h->wave_clusters < 0) return 1;
    int cap = (h->wave_clusters - n_gru / kWvCS) * kWvCS;
    if (cap > kWvMaxBatch) cap = kWvMaxBatch;
    if (cap < 1) return 1;
    int W = (int)h->opt_wave_width;
    if (W <= 0) { W = 128 / (p.batch < cap ? p.batch : cap); }     // ~128 nodes per step over the batch: two GRU passes
    if (W < 1) W = 1;
    if (W > kWvMaxW) W = kWvMaxW;
    {   // a GRU CTA keeps at most kWvMaxItems compacted items per step; a request CTA merges at most 256 new candidates
        const int nbmax = p.batch < cap ? p.batch : cap;
        if (W * nbmax > kWvMaxItems) W = kWvMaxItems / nbmax;
        if (W * p.k > 256) W = 256 / p.k;
    }
    const int e_max = h->slot_stride - 1;
    int nsl = W < kWvMaxSlices ? W : kWvMaxSlices;
    if (nsl > p.L) nsl = p.L;
    size_t rs = 0;
    for (; nsl >= 1; --nsl) {
        rs = wave_req_smem2(p.r, p.M, p.B, p.k, W, e_max, nsl);
        if (rs <= (size_t)h->max_smem_optin) break;
    }
    if (nsl < 1) return 1;
    const size_t dsm = gs > rs ? gs : rs;
    if (probe) return DT_OK;
    int rc = m_begin ? phase_mark(h, 2, st) : DT_OK;
    if (rc) return rc;
    for (int b0 = 0; b0 < p.batch; b0 += cap) {
        const int nb = (p.batch - b0 < cap) ? (p.batch - b0) : cap;
        WaveParams f;
        memset(&f, 0, sizeof(f));
        f.e = p;
        f.e.batch = nb;
        f.e.C = p.C + (size_t)b0 * p.L * p.r;
        f.e.cand_id = p.cand_id + (size_t)b0 * p.L * p.M; f.e.cand_val = p.cand_val + (size_t)b0 * p.L * p.M;
        f.e.tokens = p.tokens + (size_t)b0 * p.N; f.e.parents = p.parents + (size_t)b0 * p.N; f.e.depths = p.depths + (size_t)b0 * p.N;
        f.e.positions = p.positions + (size_t)b0 * p.N; f.e.scores = p.scores + (size_t)b0 * p.N;
        f.e.mask = p.mask + (size_t)b0 * p.N * p.N; f.e.n_nodes = p.n_nodes + b0;
        f.e.root_tokens = p.root_tokens + b0; f.e.root_positions = p.root_positions ? p.root_positions + b0 : nullptr;
        f.n_groups = h->opt_wave_groups ? (int)h->opt_wave_groups : 2;
        if (f.n_groups > nb) f.n_groups = nb;
        f.n_gru = n_gru; f.slot_stride = h->slot_stride; f.W = W; f.n_slices = nsl; f.e_max = e_max;
        f.P = n_gru / kWvCS; f.rpc = 16 * ((p.r + 16 * kWvCS - 1) / (16 * kWvCS));
        const size_t so = (size_t)b0 * h->slot_stride * p.g;
        f.s_hi = h->s_hi + so; f.s_lo = h->s_lo + so; f.s32 = h->states + so;
        f.partial = h->wv_partial + (size_t)b0 * kWvMaxW * f.P * p.r;
        f.desc = h->wv_desc + (size_t)b0 * kWvDescWords;
        f.flags = h->wv_flags; f.round_ctr = h->wv_round; f.err = h->wv_err; f.stats = (b0 == 0) ? h->wv_stats : nullptr;
        if (sel >= 0) {
            f.sched_sel = h->sched_sel; f.sched_thr = h->sched_thr; f.run_peaked = (sel == 2);
            f.W_peaked = W < 4 ? W : 4;
        }
        cudaLaunchConfig_t cfg;
        memset(&cfg, 0, sizeof(cfg));
        cfg.gridDim = dim3(n_gru + (nb + kWvCS - 1) / kWvCS * kWvCS); cfg.blockDim = dim3(kWvThreads);
        cfg.dynamicSmemBytes = dsm; cfg.stream = st;
        cudaLaunchAttribute at[2];
        at[0].id = cudaLaunchAttributeClusterDimension; at[0].val.clusterDim.x = kWvCS; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
        at[1].id = cudaLaunchAttributeCooperative; at[1].val.cooperative = 1;
        cfg.attrs = at; cfg.numAttrs = 2;
        cudaError_t e = cudaLaunchKernelEx(&cfg, wave_expand_kernel, f);
        h->launches++;
        DT_CUDA(h, e);
    }
    h->path_taken = 5;
    if (!m_end) return DT_OK;
    if ((rc = phase_mark(h, 3, st))) return rc;
    return phase_mark(h, 4, st);
}

// Depth-synchronous frontier schedule (dt_frontier.cuh): L per-depth launches + the ledger selection / emitter.
template <typename T>
static int launch_frontier(dt_handle *h, const ExpandParams &p, cudaStream_t st) {
    FrontierParams f;
    f.e = p; f.W = p.B;                              // W = B: the same node set as the heap
    f.fstate = h->fr_state; f.led_tok = h->led_tok; f.led_par = h->led_par; f.led_g = h->led_g;
    f.led_cnt = h->led_cnt; f.led_slot = h->led_slot; f.fr_ref = h->fr_ref; f.fr_plane = h->fr_plane; f.n_fr = h->fr_n;
    const size_t dsm = (size_t)(p.g + p.r + 2 * p.M + kFrLanes * p.g) * 4 + (size_t)p.M * 4;
    if (dsm > 48 * 1024) return DT_ERR_UNSUPPORTED;
    int rc = phase_mark(h, 2, st);
    if (rc) return rc;
    for (int d = 0; d < p.L; ++d) {
        frontier_depth_kernel<T><<<p.batch, kExpThreads, dsm, st>>>(f, d);
        h->launches++;
    }
    DT_CUDA(h, cudaGetLastError());
    if ((rc = phase_mark(h, 3, st))) return rc;
    frontier_finalize_kernel<<<p.batch, kExpThreads, (size_t)4 * p.N * 4, st>>>(f);
    h->launches++;
    DT_CUDA(h, cudaGetLastError());
    return phase_mark(h, 4, st);
}

// Factorized arms (dt_scorers.cuh): best-first over the per-depth menus in h->menu_*, then the emitter.
static int launch_factorized(dt_handle *h, const ExpandParams &p, cudaStream_t st) {
    ScorerParams sp;
    sp.e = p; sp.menu_tok = h->menu_tok; sp.menu_lp = h->menu_lp;
    const size_t dsm = factorized_smem(p.L, p.k, p.N);
    if (dsm > 48 * 1024) return DT_ERR_UNSUPPORTED;
    factorized_expand_kernel<<<p.batch, kFusThreads, dsm, st>>>(sp);
    h->launches++;
    DT_CUDA(h, cudaGetLastError());
    int rc = phase_mark(h, 3, st);
    if (rc) return rc;
    return phase_mark(h, 4, st);
}

template <typename T>
static int launch_expansion(dt_handle *h, ExpandParams &p, cudaStream_t st) {
    const int g = p.g;
    init_round_kernel<<<p.batch, 32, 0, st>>>(p);
    root_state_kernel<<<p.batch, 256, 0, st>>>(h->P, p.root_tokens, g, p.V, p.states, (long long)p.N * g);
    h->launches += 2;
    int rc = phase_mark(h, 2, st);
    if (rc) return rc;
    const size_t dsm = (size_t)(g + p.r + p.M) * 4 + (size_t)p.M * 4;   // opt-in above 48 KB done in dt_create
    const int gru_grid = (g + kGruUnitsPerCta - 1) / kGruUnitsPerCta;
    for (int t = 0; t < p.B; ++t) {
        if (t > 0) { gru_step_kernel<T><<<gru_grid, kExpThreads, 0, st>>>(p, t); h->launches++; }
        expand_kernel<T><<<p.batch, kExpThreads, dsm, st>>>(p, t);
        h->launches++;
    }
    if ((rc = phase_mark(h, 3, st))) return rc;
    emit_kernel<<<p.batch, kExpThreads, 0, st>>>(p);
    h->launches++;
    DT_CUDA(h, cudaGetLastError());
    return phase_mark(h, 4, st);
}

extern "C" int dt_build_trees(dt_handle *h, const void *marginal_logits, const void *backbone_hidden,
                              const int32_t *root_tokens, const int32_t *root_positions, int32_t batch,
                              int32_t M, int32_t B, float temperature, const dt_outputs *out, void *stream) {
    if (!h || !out) return DT_ERR_INVALID_ARG;
    if (batch < 0 || batch > h->max_batch) return DT_ERR_INVALID_ARG;
    if (M < h->k || M > h->max_M || B < 1 || B > h->max_B) return DT_ERR_INVALID_ARG;
    if (!(temperature >= 0.0f) || isinf(temperature)) return DT_ERR_INVALID_ARG;
    h->launches = 0;
    if (batch == 0) return DT_OK;               // empty batch: nothing to read or write
    if (!marginal_logits || !backbone_hidden || !root_tokens) return DT_ERR_INVALID_ARG;
    if (!out->tokens || !out->parents || !out->depths || !out->positions || !out->scores || !out->mask || !out->n_nodes)
        return DT_ERR_INVALID_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    const dt_weights &w = h->w;
    const int rows = batch * h->L;

    int rc = phase_mark(h, 0, st);
    if (rc) return rc;
    // C = H W1[:, 0:d]^T   (Fact B PAPER.md:83-89).  bf16: tensor cores.
    const bool mma = h->mma_ok && ((reinterpret_cast<uintptr_t>(backbone_hidden) & 15u) == 0) &&
                     rows <= h->max_batch * h->L;
    // bf16: tensor cores, forked onto the handle's side stream so it overlaps the HBM-bound select (fork/join by
    // events: capture-safe, becomes a parallel graph branch).  Measured at C5: overlapped select + GEMM 64 us,
    // back to back 51 + 35 us.
    const bool serial = mma && h->opt_gemm_serial;
    if (mma && !serial) {
        DT_CUDA(h, cudaEventRecord(h->ev_fork, st));
        DT_CUDA(h, cudaStreamWaitEvent(h->side, h->ev_fork, 0));
        rc = (h->tcg_ok && h->opt_gemm != 1)
            ? launch_gemm_tc(h, backbone_hidden, w.d, w.corr_w1, (long long)w.d + w.g, h->C, w.r, rows, w.r, w.d, h->side)
            : launch_gemm_mma(h, backbone_hidden, w.d, w.corr_w1, (long long)w.d + w.g, h->C, w.r, rows, w.r, w.d, h->side);
        if (rc) return rc;
        DT_CUDA(h, cudaEventRecord(h->ev_join, h->side));
    }
    rc = launch_select(h, marginal_logits, rows, M, h->cand_id, h->cand_val, st);
    if (rc) return rc;
    if ((rc = phase_mark(h, 1, st))) return rc;
    if (serial) {
        rc = (h->tcg_ok && h->opt_gemm != 1)
            ? launch_gemm_tc(h, backbone_hidden, w.d, w.corr_w1, (long long)w.d + w.g, h->C, w.r, rows, w.r, w.d, st)
            : launch_gemm_mma(h, backbone_hidden, w.d, w.corr_w1, (long long)w.d + w.g, h->C, w.r, rows, w.r, w.d, st);
    } else if (mma) DT_CUDA(h, cudaStreamWaitEvent(st, h->ev_join, 0));
    else if (w.dtype == DT_BF16)
        rc = launch_gemm_nt<__nv_bfloat16>(h, backbone_hidden, w.d, w.corr_w1, (long long)w.d + w.g, h->C, w.r, rows, w.r, w.d, st);
    else
        rc = launch_gemm_nt<float>(h, backbone_hidden, w.d, w.corr_w1, (long long)w.d + w.g, h->C, w.r, rows, w.r, w.d, st);
    if (rc) return rc;

    ExpandParams p;
    memset(&p, 0, sizeof(p));
    p.w_hh = w.gru_w_hh; p.w1 = w.corr_w1; p.w2 = w.corr_w2; p.P = h->P;
    p.V = w.V; p.d = w.d; p.g = w.g; p.r = w.r;
    p.batch = batch; p.L = h->L; p.M = M; p.B = B; p.k = h->k; p.N = B + 1;
    p.T_eff = (temperature == 0.0f) ? 1.0f : temperature;          // reading A7
    p.C = h->C; p.cand_id = h->cand_id; p.cand_val = h->cand_val;
    p.states = h->states; p.heap_g = h->heap_g; p.heap_tp = h->heap_tp; p.heap_cnt = h->heap_cnt;
    p.heap_cap = h->heap_cap;
    p.tokens = out->tokens; p.parents = out->parents; p.depths = out->depths; p.positions = out->positions;
    p.n_nodes = out->n_nodes; p.scores = out->scores; p.mask = out->mask;
    p.root_tokens = root_tokens; p.root_positions = root_positions;
    if (h->opt_schedule == 1 && h->opt_scorer == 0) {   // frontier schedule of the DominoTree scorer
        // bf16: the frontier's per-depth GEMM over many nodes of many requests IS the wavefront kernel's GRU pass; at its
        // maximal width a step expands every unexpanded member of the top-B frontier (up to 15 per request), on tcgen05.
        // Shapes the wavefront kernel rejects (and fp32) take the depth-synchronous ledger kernels (warp FMA).
        if (w.dtype == DT_BF16 && h->opt_expand_path == 0) {
            const int64_t keep = h->opt_wave_width;
            h->opt_wave_width = kWvMaxW;
            h->opt_expand_path = 5;
            rc = launch_wave(h, p, st);
            h->opt_wave_width = keep;
            h->opt_expand_path = 0;
            if (rc <= 0) return rc;
        }
        return (w.dtype == DT_BF16) ? launch_frontier<__nv_bfloat16>(h, p, st) : launch_frontier<float>(h, p, st);
    }
    if (h->opt_scorer == 1) {                       // Marg: menus from the base logits alone, no GRU, no C
        ScorerParams sp;
        sp.e = p; sp.menu_tok = h->menu_tok; sp.menu_lp = h->menu_lp;
        marg_menu_kernel<<<rows, 256, 0, st>>>(sp);
        h->launches++;
        DT_CUDA(h, cudaGetLastError());
        if ((rc = phase_mark(h, 2, st))) return rc;
        return launch_factorized(h, p, st);
    }
    if (h->opt_scorer == 2) {                       // Cond-static: corrected menus along the greedy chain
        if (w.dtype != DT_BF16) return DT_ERR_UNSUPPORTED;
        ExpandParams ps = p;
        ps.B = h->L; ps.N = h->L + 1;               // the chain has L nodes below the root; outputs are not touched
        rc = launch_fused(h, ps, st, true);
        if (rc > 0) return DT_ERR_UNSUPPORTED;      // shape the fused kernel rejects
        if (rc) return rc;
        return launch_factorized(h, p, st);
    }
    h->path_taken = 1;
    if (w.dtype == DT_BF16) {
        // adaptive round: both persistent kernels are enqueued, the device's schedule word lets one of them run
        if (h->opt_expand_path == 0 && h->opt_adaptive && launch_wave(h, p, st, -1, true) == DT_OK &&
            launch_fused(h, p, st, false, -1, true) == DT_OK) {
            DT_CUDA(h, cudaMemsetAsync(h->sched_sel, 0, 4, st));
            h->sched_thr = (unsigned int)(0.6 * 65536.0 * rows);
            wave_regime_kernel<<<(rows + 7) / 8, 256, 0, st>>>(h->cand_val, rows, M, 1.0f / p.T_eff, h->sched_sel);
            h->launches++;
            DT_CUDA(h, cudaGetLastError());
            // chains longer than ~48 nodes: even a peaked round pays in the wavefront kernel (at a width of 4); shorter ones
            // go to the lock-step kernel, whose step is shorter
            const bool wave_only = B >= 48;
            rc = launch_wave(h, p, st, wave_only ? 2 : 1, false, true, wave_only);
            if (rc) return rc < 0 ? rc : DT_ERR_CUDA;
            if (!wave_only) {
                const int64_t n = h->launches;
                rc = launch_fused(h, p, st, false, 0, false, false, true);
                h->launches = n + 1;
            }
            h->path_taken = 6;
            return rc < 0 ? rc : (rc ? DT_ERR_CUDA : DT_OK);
        }
        rc = launch_wave(h, p, st);
        if (rc <= 0) return rc;
        rc = launch_fused(h, p, st);
        if (rc <= 0) return rc;
        return launch_expansion<__nv_bfloat16>(h, p, st);
    }
    return launch_expansion<float>(h, p, st);
}

extern "C" int dt_adaptive_budget(dt_handle *h, const dt_outputs *tree, int32_t batch, int32_t B, double C_d, const float *cv,
                                  int32_t *n_star, float *phi, void *stream) {
    if (!h || !tree) return DT_ERR_INVALID_ARG;
    if (batch < 0 || batch > h->max_batch || B < 1 || B > h->max_B || !(C_d >= 0.0) || isinf(C_d)) return DT_ERR_INVALID_ARG;
    h->launches = 0;
    if (batch == 0) return DT_OK;
    if (!tree->scores || !tree->n_nodes || !cv || !n_star) return DT_ERR_INVALID_ARG;
    adaptive_budget_kernel<<<(batch + 63) / 64, 64, 0, (cudaStream_t)stream>>>(tree->scores, tree->n_nodes, B + 1, batch, C_d, cv,
                                                                               n_star, phi);
    h->launches++;
    DT_CUDA(h, cudaGetLastError());
    return DT_OK;
}

extern "C" int dt_commit_paths(dt_handle *h, const dt_outputs *tree, int32_t batch, int32_t B, const int32_t *target_next,
                               const uint8_t *edge_ok, int32_t *accept_len, int32_t *path_slots, int32_t *bonus_token,
                               void *stream) {
    if (!h || !tree) return DT_ERR_INVALID_ARG;
    if (batch < 0 || batch > h->max_batch || B < 1 || B > h->max_B) return DT_ERR_INVALID_ARG;
    if ((target_next != nullptr) == (edge_ok != nullptr)) return DT_ERR_INVALID_ARG;
    h->launches = 0;
    if (batch == 0) return DT_OK;
    if (!tree->tokens || !tree->parents || !tree->depths || !tree->scores || !tree->n_nodes || !accept_len || !path_slots)
        return DT_ERR_INVALID_ARG;
    CommitParams c;
    c.tokens = tree->tokens; c.parents = tree->parents; c.depths = tree->depths; c.n_nodes = tree->n_nodes;
    c.scores = tree->scores; c.target_next = target_next; c.edge_ok = edge_ok;
    c.accept_len = accept_len; c.path_slots = path_slots; c.bonus_token = bonus_token;
    c.N = B + 1; c.L = h->L;
    commit_paths_kernel<<<batch, 256, 0, (cudaStream_t)stream>>>(c);
    h->launches++;
    DT_CUDA(h, cudaGetLastError());
    return DT_OK;
}

extern "C" int dt_tree_links(dt_handle *h, const dt_outputs *tree, int32_t batch, int32_t B, int32_t *first_child,
                             int32_t *next_sibling, void *stream) {
    if (!h || !tree) return DT_ERR_INVALID_ARG;
    if (batch < 0 || batch > h->max_batch || B < 1 || B > h->max_B) return DT_ERR_INVALID_ARG;
    h->launches = 0;
    if (batch == 0) return DT_OK;
    if (!tree->parents || !tree->n_nodes || !first_child || !next_sibling) return DT_ERR_INVALID_ARG;
    tree_links_kernel<<<batch, 256, 0, (cudaStream_t)stream>>>(tree->parents, tree->n_nodes, B + 1, first_child, next_sibling);
    h->launches++;
    DT_CUDA(h, cudaGetLastError());
    return DT_OK;
}

extern "C" int dt_build_trees_host(dt_handle *h, const void *logits_h, const void *hidden_h,
                                   const int32_t *roots_h, const int32_t *rpos_h, int32_t batch,
                                   int32_t M, int32_t B, float temperature, const dt_outputs *oh, void *stream) {
    if (!h || !oh) return DT_ERR_INVALID_ARG;
    if (batch < 0 || batch > h->max_batch || B < 1 || B > h->max_B) return DT_ERR_INVALID_ARG;
    if (batch == 0) return DT_OK;
    if (!logits_h || !hidden_h || !roots_h) return DT_ERR_INVALID_ARG;
    if (!oh->tokens || !oh->parents || !oh->depths || !oh->positions || !oh->scores || !oh->mask || !oh->n_nodes)
        return DT_ERR_INVALID_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    const size_t N = (size_t)h->max_B + 1;
    if (!h->stage) {                            // sized for the handle's maxima, allocated once
        size_t off = 0;
        auto carve = [&](size_t bytes) { size_t o = off; off = align_up(off + bytes, 256); return o; };
        carve((size_t)h->max_batch * h->L * h->w.V * h->esize);
        carve((size_t)h->max_batch * h->L * h->w.d * h->esize);
        carve((size_t)h->max_batch * 4); carve((size_t)h->max_batch * 4);
        carve((size_t)h->max_batch * N * 4 * 5); carve((size_t)h->max_batch * N * N); carve((size_t)h->max_batch * 4);
        if (cudaMalloc(&h->stage, off) != cudaSuccess) { cudaGetLastError(); h->stage = nullptr; return DT_ERR_ALLOC; }
        h->stage_bytes = off;
    }
    size_t off = 0;
    auto carve = [&](size_t bytes) { char *q = h->stage + off; off = align_up(off + bytes, 256); return q; };
    const size_t lb = (size_t)batch * h->L * h->w.V * h->esize, hb = (size_t)batch * h->L * h->w.d * h->esize;
    char *d_logits = carve((size_t)h->max_batch * h->L * h->w.V * h->esize);
    char *d_hidden = carve((size_t)h->max_batch * h->L * h->w.d * h->esize);
    int32_t *d_roots = (int32_t *)carve((size_t)h->max_batch * 4);
    int32_t *d_rpos = (int32_t *)carve((size_t)h->max_batch * 4);
    char *d_i32 = carve((size_t)h->max_batch * N * 4 * 5);
    uint8_t *d_mask = (uint8_t *)carve((size_t)h->max_batch * N * N);
    int32_t *d_nn = (int32_t *)carve((size_t)h->max_batch * 4);
    const size_t Nb = (size_t)B + 1, slab = (size_t)batch * Nb * 4;
    dt_outputs od;
    od.tokens = (int32_t *)(d_i32); od.parents = (int32_t *)(d_i32 + slab); od.depths = (int32_t *)(d_i32 + 2 * slab);
    od.positions = (int32_t *)(d_i32 + 3 * slab); od.scores = (float *)(d_i32 + 4 * slab);
    od.mask = d_mask; od.n_nodes = d_nn;
    DT_CUDA(h, cudaMemcpyAsync(d_logits, logits_h, lb, cudaMemcpyHostToDevice, st));
    DT_CUDA(h, cudaMemcpyAsync(d_hidden, hidden_h, hb, cudaMemcpyHostToDevice, st));
    DT_CUDA(h, cudaMemcpyAsync(d_roots, roots_h, (size_t)batch * 4, cudaMemcpyHostToDevice, st));
    if (rpos_h) DT_CUDA(h, cudaMemcpyAsync(d_rpos, rpos_h, (size_t)batch * 4, cudaMemcpyHostToDevice, st));
    int rc = dt_build_trees(h, d_logits, d_hidden, d_roots, rpos_h ? d_rpos : nullptr, batch, M, B, temperature, &od, st);
    if (rc) return rc;
    DT_CUDA(h, cudaMemcpyAsync(oh->tokens, od.tokens, slab, cudaMemcpyDeviceToHost, st));
    DT_CUDA(h, cudaMemcpyAsync(oh->parents, od.parents, slab, cudaMemcpyDeviceToHost, st));
    DT_CUDA(h, cudaMemcpyAsync(oh->depths, od.depths, slab, cudaMemcpyDeviceToHost, st));
    DT_CUDA(h, cudaMemcpyAsync(oh->positions, od.positions, slab, cudaMemcpyDeviceToHost, st));
    DT_CUDA(h, cudaMemcpyAsync(oh->scores, od.scores, slab, cudaMemcpyDeviceToHost, st));
    DT_CUDA(h, cudaMemcpyAsync(oh->mask, od.mask, (size_t)batch * Nb * Nb, cudaMemcpyDeviceToHost, st));
    DT_CUDA(h, cudaMemcpyAsync(oh->n_nodes, od.n_nodes, (size_t)batch * 4, cudaMemcpyDeviceToHost, st));
    DT_CUDA(h, cudaStreamSynchronize(st));
    return DT_OK;
}

// ------------------------------------------------------------------------------------------------------------------
// dt_select_topm_static: the top-M select (a1) for callers that cannot allocate -- no handle, no cudaMalloc / cudaFree, no
// allocating library call.  The select kernels need scratch (per-row arrival tickets and shared thresholds, per-chunk
// partial lists when a row is split into chunks); here it lives in ONE file-scope device array that every GPU which
// loads the library holds until exit: 8 KiB of tickets / thresholds + 2 MiB of partials.  Every call shares it and it
// keeps the last call's contents: the tickets and thresholds are cleared on `stream` in front of every launch, the
// partials are written before they are read.  Two calls that overlap on the GPU (different streams, or graphs replayed
// concurrently) race on it.
constexpr int kStaticMaxRows = DT_STATIC_MAX_ROWS;
constexpr size_t kStaticPartKeys = (size_t)DT_STATIC_PART_BYTES / 8;
constexpr size_t kStaticCtlWords = 2 * (size_t)kStaticMaxRows * 4 / 8;      // u64 words of the ticket + threshold arrays
static __device__ __align__(256) unsigned long long g_static_scratch[kStaticCtlWords + kStaticPartKeys];

namespace {
struct StaticDev { bool tried = false; int rc = DT_OK; unsigned long long *scratch = nullptr; int sms = 0; bool bulk_ok = false; };
constexpr int kStaticMaxDev = 64;
StaticDev g_static_dev[kStaticMaxDev];
std::mutex g_static_mu;

// Once per device, with that device current: in host code `g_static_scratch` is a host-side stand-in, not a device
// address; the kernel gets what cudaGetSymbolAddress returns for the current device.
int static_setup(int dev, StaticDev **out) {
    if (dev < 0 || dev >= kStaticMaxDev) return DT_ERR_UNSUPPORTED;
    std::lock_guard<std::mutex> lk(g_static_mu);
    StaticDev &d = g_static_dev[dev];
    if (!d.tried) {
        d.tried = true;
        void *ptr = nullptr;
        if (cudaGetSymbolAddress(&ptr, g_static_scratch) != cudaSuccess || !ptr ||
            cudaDeviceGetAttribute(&d.sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || d.sms < 1) {
            cudaGetLastError();
            d.rc = DT_ERR_CUDA;
        } else {
            d.scratch = reinterpret_cast<unsigned long long *>(ptr);
            d.bulk_ok =
                cudaFuncSetAttribute(select_topm_bulk_kernel<__nv_bfloat16, SelectSmemBig>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sel_bulk_dyn_smem<SelectSmemBig>()) == cudaSuccess &&
                cudaFuncSetAttribute(select_topm_bulk_kernel<float, SelectSmemBig>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sel_bulk_dyn_smem<SelectSmemBig>()) == cudaSuccess;
            if (!d.bulk_ok) cudaGetLastError();
        }
    }
    *out = &d;
    return d.rc;
}
}  // namespace

extern "C" int dt_static_init(void) {
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) { cudaGetLastError(); return DT_ERR_CUDA; }
    StaticDev *d = nullptr;
    return static_setup(dev, &d);
}

extern "C" int dt_select_topm_static(const void *logits, int32_t dtype, int32_t rows, int32_t V, int32_t M,
                                     int32_t *cand_id, float *cand_val, void *stream) {
    if (dtype != DT_BF16 && dtype != DT_F32) return DT_ERR_INVALID_ARG;
    if (rows < 0 || V < 1 || M < 1 || M > V) return DT_ERR_INVALID_ARG;
    if (rows > kStaticMaxRows || M > DT_MAX_M) return DT_ERR_STATIC_LIMIT;
    if (rows == 0) return DT_OK;
    if (!logits || !cand_id || !cand_val) return DT_ERR_INVALID_ARG;
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) { cudaGetLastError(); return DT_ERR_CUDA; }
    StaticDev *d = nullptr;
    int rc = static_setup(dev, &d);
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    const int kvec = (dtype == DT_BF16) ? 8 : 4;
    const bool aligned = (V % kvec == 0) && ((reinterpret_cast<uintptr_t>(logits) & 15u) == 0);
    const bool bulk = aligned && d->bulk_ok;
    SelectParams p;
    p.logits = logits; p.rows = rows; p.V = V; p.M = M;
    p.row_vecs = (V + kvec - 1) / kvec;
    // chunks per row: enough CTAs to fill the GPU, chunks long enough to keep a CTA's warps busy, the merging CTA's
    // buffer holds S * M keys, and all partial lists fit the static array (S = 1 needs none)
    int S = (3 * d->sms + rows - 1) / rows;
    const int by_len = p.row_vecs / 4096 < 1 ? 1 : p.row_vecs / 4096;
    if (S > by_len) S = by_len;
    if (S > SelectSmemBig::kCap / M) S = SelectSmemBig::kCap / M;
    if (S > kSelMaxChunks) S = kSelMaxChunks;
    while (S > 1 && (size_t)rows * S * M > kStaticPartKeys) --S;
    if (S < 1) S = 1;
    p.S = S;
    p.chunk_vecs = (p.row_vecs + S - 1) / S;
    if (bulk) p.chunk_vecs = (p.chunk_vecs + kSelTileVecs - 1) / kSelTileVecs * kSelTileVecs;
    p.cand_id = cand_id; p.cand_val = cand_val;
    p.row_counter = reinterpret_cast<unsigned int *>(d->scratch);
    p.row_tau = p.row_counter + kStaticMaxRows;
    p.part = d->scratch + kStaticCtlWords;
    p.span = nullptr;
    // the array keeps the previous call's contents: tickets and thresholds must start at zero
    if (cudaMemsetAsync(d->scratch, 0, kStaticCtlWords * 8, st) != cudaSuccess) { cudaGetLastError(); return DT_ERR_CUDA; }
    const dim3 grid(S, rows);
    if (bulk) {
        if (dtype == DT_BF16) select_topm_bulk_kernel<__nv_bfloat16, SelectSmemBig><<<grid, 256, sel_bulk_dyn_smem<SelectSmemBig>(), st>>>(p);
        else select_topm_bulk_kernel<float, SelectSmemBig><<<grid, 256, sel_bulk_dyn_smem<SelectSmemBig>(), st>>>(p);
    } else if (dtype == DT_BF16) {
        if (aligned) select_topm_kernel<__nv_bfloat16, true><<<grid, kSelThreads, 0, st>>>(p);
        else select_topm_kernel<__nv_bfloat16, false><<<grid, kSelThreads, 0, st>>>(p);
    } else {
        if (aligned) select_topm_kernel<float, true><<<grid, kSelThreads, 0, st>>>(p);
        else select_topm_kernel<float, false><<<grid, kSelThreads, 0, st>>>(p);
    }
    if (cudaGetLastError() != cudaSuccess) return DT_ERR_CUDA;
    return DT_OK;
}

#ifdef DT_TRACE
// measurement builds only (libdominotree_trace.so, -DDT_TRACE): copy the in-kernel timeline of the last wavefront round
// to `host` (2 roles x kWvTraceSteps x kWvTraceStamps u64 of %globaltimer, zero = not reached) and clear it
extern "C" int dt_trace_read(unsigned long long *host) {
    const size_t n = sizeof(unsigned long long) * 2 * dt::kWvTraceSteps * dt::kWvTraceStamps;
    if (cudaDeviceSynchronize() != cudaSuccess) return DT_ERR_CUDA;
    if (cudaMemcpyFromSymbol(host, dt::g_wv_trace, n) != cudaSuccess) return DT_ERR_CUDA;
    void *sym = nullptr;
    if (cudaGetSymbolAddress(&sym, dt::g_wv_trace) != cudaSuccess || cudaMemset(sym, 0, n) != cudaSuccess) return DT_ERR_CUDA;
    return DT_OK;
}
#endif

/* lst.h -- C ABI of the B200-native Line Segment Tracking (LST) object-building chain.
 *
 * What it computes (arxiv 2407.18231, PAPER.md):
 *   outer-tracker hits --[two sensors of a module]--> Mini-Doublets (MD)
 *   MD x MD on modules joined by the precomputed connection map --> Line Segments
 *   LS x LS sharing an MD --> T3;  T3 x T3 sharing an MD --> T5
 *   inner-tracker seeds (pLS) x T3 / T5 --> pT3 / pT5
 *   duplicate removal + selection of {pT5, pT3, T5, unlinked pLS} track candidates
 * The numeric selections (deferred by PAPER.md:29 to its Refs. [4], [5]) are the documented
 * stand-in of CUTS.md; all cut arithmetic is binary32, fixed order, no FMA.
 *
 * Conventions
 *   - All functions return 0 (LST_OK) or a negative lst_status; no exception crosses the ABI.
 *   - "host" / "device" is stated per pointer.  Inputs are caller-owned and never retained past the
 *     call that takes them (lst_ctx_run: past the following lst_ctx_sync).  Outputs are library-owned
 *     until lst_free.
 *   - Indices in outputs: hit indices refer to the caller's INPUT hit order within the event
 *     (0-based, event-local); object indices (md, ls, t3, t5, pls) are event-local positions in the
 *     returned arrays of that event.
 *   - Overflow of a preallocated object array returns LST_ERR_CAPACITY; nothing is ever truncated.
 *   - One lst_ctx per CUDA stream; a lst_geometry is immutable and may be shared by many contexts.
 */
#ifndef LST_H
#define LST_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum lst_status {
  LST_OK = 0,
  LST_ERR_ARG = -1,      /* NULL / negative size / sensor id or event offsets out of range */
  LST_ERR_CUDA = -2,     /* CUDA runtime error (no device, out of memory, launch failure) */
  LST_ERR_CAPACITY = -3, /* an object array of the context is too small for this batch */
  LST_ERR_GEOMETRY = -4, /* malformed module table or connection map */
  LST_ERR_LIMIT = -5     /* size beyond the fixed maximum of an entry point that cannot allocate */
} lst_status;

/* Static string for a status code. */
const char* lst_strerror(int status);

/* One module = one tile of a layer with its two sensors; sensor ids are 2*m (lower)
 * and 2*m+1 (upper).  Only `subdet` enters the arithmetic (CUTS.md 3, 4); the rest is carried. */
typedef struct lst_module {
  int32_t subdet; /* 0 = barrel, 1 = endcap */
  int32_t layer;  /* 1..6 barrel layer, 1..5 endcap disk */
  int32_t side;   /* 0 barrel, -1 / +1 endcap side */
  int32_t ring;   /* barrel z-tile / endcap ring */
} lst_module;

/* Cut constants of CUTS.md section 1 (same order) and the stage mask of CUTS.md section 9. */
typedef struct lst_params {
  float b_field, pt_min, z0_max;
  float md_b_phi_tol, md_z_tol, md_e_slope, md_e_tol;
  float ls_kappa_max, ls_z_tol, ls_dir_tol;
  float t3_kappa_max, t3_z_tol0, t3_z_tol1;
  float t5_tol0, t5_tol1;
  float pt_gate_tol, pt_k_tol0, pt_k_tol1, pt_z_tol;
  float near_rel; /* NEAR_REL of CUTS.md section 0; 0 <= near_rel <= 1e-5 (the default), else lst_load_geometry
                     returns LST_ERR_ARG: the kernels' pre-filters are sized for a near window of at most 1e-5 */
  int32_t stage_mask; /* bit0 MD, 1 LS, 2 T3, 3 T5, 4 pT3/pT5, 5 duplicate removal + TC, 6 T4, 7 learned T5 */
  /* extensions of CUTS.md sections 10 and 11, used only with stage_mask bits 6 / 7 */
  float t4_tol0, t4_tol1;
  float t5_mlp_scale, t5_mlp_thr;
  float t5_mlp[65]; /* W1[8][6] row-major, b1[8], W2[8], b2 */
} lst_params;

/* Fills *p with the defaults of CUTS.md section 1 (stage_mask = 0x3f). */
void lst_default_params(lst_params* p);

/* Capacities of one context (object counts summed over the events of a batch).  max_md may not exceed
 * LST_MAX_MD (the Line-Segment stage packs an MD index and two flags into one 32-bit word): lst_ctx_create
 * returns LST_ERR_ARG. */
#define LST_MAX_MD (1 << 27)
typedef struct lst_caps {
  int32_t max_events;
  int32_t max_hits, max_pls;
  int32_t max_md, max_ls, max_t3, max_t5, max_pt3, max_pt5, max_tc;
  int32_t max_t4; /* T4 objects (CUTS.md section 10; only used with stage_mask bit 6) */
} lst_caps;

/* Defaults sized for 16 PU250-like events (a few hundred MB; the B200 has 180 GB). */
void lst_default_caps(lst_caps* c);
/* Device bytes a context with these capacities allocates for a geometry of n_modules. */
size_t lst_workspace_bytes(const lst_caps* c, int32_t n_modules);

/* Outer-tracker hits of a batch, structure of arrays.  x, y, z in cm. */
typedef struct lst_hits {
  const float* x;
  const float* y;
  const float* z;
  const int32_t* sensor;        /* 2*module + {0,1}; with sensor_u16 != 0 the array holds uint16_t instead */
  int32_t n;                    /* hits in the batch */
  const int32_t* event_offsets; /* HOST pointer, n_events+1 entries, [0] = 0, [n_events] = n;
                                   NULL = one event */
  int32_t on_device;            /* 0: x, y, z, sensor are host pointers; 1: device pointers */
  int32_t sensor_u16;           /* != 0: `sensor` points to uint16_t ids (14 instead of 16 bytes per hit over PCIe);
                                   needs 2 * n_modules <= 65536, else LST_ERR_ARG */
} lst_hits;

/* Inner-tracker seeds (pLS) of a batch (reading S6 of DESIGN.md). */
typedef struct lst_pls {
  const float* pt;  /* GeV */
  const int32_t* q; /* +-1 */
  const float *x0, *y0, *z0; /* inner pixel hit */
  const float *x1, *y1, *z1; /* outer pixel hit */
  int32_t n;
  const int32_t* event_offsets; /* HOST pointer, n_events+1 entries; NULL = one event */
  int32_t on_device;
} lst_pls;

typedef struct lst_geometry lst_geometry;
typedef struct lst_ctx lst_ctx;

enum { LST_ST_MD = 0, LST_ST_LS, LST_ST_T3, LST_ST_T5, LST_ST_PT3, LST_ST_PT5, LST_ST_T4, LST_N_STAGES };

/* Result of one event, host memory, library-owned (lst_free).  Layouts as in CUTS.md. */
typedef struct lst_event_out {
  uint64_t magic;
  int32_t n_md, n_ls, n_t3, n_t5, n_pt3, n_pt5, n_tc;
  int64_t near[LST_N_STAGES];    /* near-threshold candidates of THIS event per stage (CUTS.md section 0) */
  int64_t n_tests[LST_N_STAGES]; /* candidates of THIS event per stage (CUTS.md sections 3-7) */
  int32_t* md_hits;   /* [n_md][2]  h_lo, h_hi (input hit indices) */
  int32_t* md_module; /* [n_md] */
  float* md_f;        /* [n_md][6]  anchor x, y, z, r and unit direction ux, uy */
  int32_t* ls_md;     /* [n_ls][2]  md_in, md_out */
  float* ls_kappa;    /* [n_ls] */
  int32_t* t3_ls;     /* [n_t3][2] */
  int32_t* t3_md;     /* [n_t3][3] */
  float* t3_k;        /* [n_t3] */
  int32_t* t5_t3;     /* [n_t5][2] */
  int32_t* t5_md;     /* [n_t5][5] */
  float* t5_score;    /* [n_t5] */
  int32_t* pt3;       /* [n_pt3][2] pls, t3 */
  float* pt3_score;
  int32_t* pt5;       /* [n_pt5][2] pls, t5 */
  float* pt5_score;
  int32_t* tc;        /* [n_tc][16] type, pls, t5, t3, hit_idx[12]; classes in order pT5, pT3, T5, pLS (, T4) */
  /* extension (CUTS.md section 10): 4-MD objects, empty unless stage_mask bit 6 is set */
  int32_t n_t4;
  int32_t* t4_t3;     /* [n_t4][2] */
  int32_t* t4_md;     /* [n_t4][4] */
  float* t4_score;    /* [n_t4] */
} lst_event_out;

/* Totals of the last batch of a context (host struct filled by lst_ctx_sync); near / n_tests are the
 * sums of the per-event counters that lst_ctx_fetch_event returns. */
typedef struct lst_batch_summary {
  int32_t n_events;
  int32_t n_hits, n_pls;
  int32_t n_md, n_ls, n_t3, n_t5, n_pt3, n_pt5, n_tc, n_t4;
  int64_t near[LST_N_STAGES];
  int64_t n_tests[LST_N_STAGES];
} lst_batch_summary;

/* ---- the three calls of north_star ---------------------------------------------------------- */

/* Copies the module table and the CSR connection map to the device.
 * modules: host, n_modules records.  conn_offsets: host, n_modules+1, [0] = 0, non-decreasing.
 * conn_targets: host, conn_offsets[n_modules] module indices.  params: host or NULL (defaults).
 * *out: library-owned, immutable; release with lst_free. */
int lst_load_geometry(const lst_module* modules, int32_t n_modules, const int32_t* conn_offsets,
                      const int32_t* conn_targets, const lst_params* params, lst_geometry** out);

/* Runs the whole chain on ONE event, synchronously, on an internal context (default capacities,
 * default stream) and returns every object array on the host.  seeds may be NULL.
 * hits->event_offsets / seeds->event_offsets must be NULL.  *out: release with lst_free.
 * Thread-safe: concurrent calls on one geometry are serialised by the library (one internal
 * context per geometry); use one lst_ctx per thread / stream for concurrency. */
int lst_run_event(lst_geometry* g, const lst_hits* hits, const lst_pls* seeds, lst_event_out** out);

/* Releases a lst_geometry, lst_ctx or lst_event_out (NULL is a no-op). */
void lst_free(void* geometry_ctx_or_event_out);

/* ---- batch / stream helpers (same chain, many events per launch sequence) ------------------- */

/* Creates a context: preallocated device workspace + the CUDA stream it launches on.
 * caps: host or NULL (defaults).  cuda_stream: a cudaStream_t / CUstream handle as void*
 * (NULL = the legacy default stream). */
int lst_ctx_create(lst_geometry* g, const lst_caps* caps, void* cuda_stream, lst_ctx** out);

/* Enqueues the chain for n_events events on the context's stream and returns without waiting.
 * Host input pointers are copied with cudaMemcpyAsync inside this call sequence (page-locked memory
 * makes that asynchronous); device input pointers are read in place.  seeds may be NULL. */
int lst_ctx_run(lst_ctx* ctx, int32_t n_events, const lst_hits* hits, const lst_pls* seeds);

/* Waits for the last lst_ctx_run, reads back the counters (a few hundred bytes) and reports
 * LST_ERR_CAPACITY / LST_ERR_ARG detected on the device.  summary may be NULL. */
int lst_ctx_sync(lst_ctx* ctx, lst_batch_summary* summary);

/* After lst_ctx_sync: copies every object array of event `event` of the last batch to the host. */
int lst_ctx_fetch_event(lst_ctx* ctx, int32_t event, lst_event_out** out);

/* After lst_ctx_sync: copies the track candidates of the whole batch to caller-owned HOST buffers.
 * tc: [cap_tc][16] int32; tc_event_offsets: n_events+1 int32.  Returns LST_ERR_CAPACITY if the
 * batch holds more than cap_tc candidates. */
int lst_ctx_fetch_tc(lst_ctx* ctx, int32_t* tc, int32_t cap_tc, int32_t* tc_event_offsets);

/* How much of the GPU one kernel of this context may occupy: `blocks` = resident 256-thread blocks per SM
 * (1..8; 0 = the default, 8: every kernel fills the GPU, best for a context that runs alone, e.g.
 * lst_run_event).  Every kernel of the chain is a persistent ticket / grid-stride loop, so the grid size
 * changes no result, only who shares the SMs: with several contexts in flight on different streams
 * (PAPER.md:79 ran 2 streams; BASELINE.json configs[4] "pipelined over CUDA streams") kernels of different
 * batches co-reside and hide each other's latency when each takes 1-2 blocks per SM.  May be called
 * between batches (the captured launch sequence is rebuilt; a batch still in flight is waited for first).  Returns LST_ERR_ARG for blocks outside 0..8. */
int lst_ctx_set_blocks_per_sm(lst_ctx* ctx, int32_t blocks);

/* How lst_ctx_run launches the chain.  enable != 0 (the default for a context on a stream of the caller's): the
 * launch sequence is captured once as a CUDA graph and replayed per batch; enable == 0: the kernels are launched
 * one by one (what a context on the legacy default stream, which cannot be captured, always does).  Same
 * kernels, same results.  Returns LST_ERR_ARG for enable != 0 on a context of the legacy default stream. */
int lst_ctx_set_graph(lst_ctx* ctx, int32_t enable);

/* Per-kernel device times of the last batch, measured with CUDA events on the context's stream.
 * enable != 0 switches the recording on for the following lst_ctx_run calls. */
int lst_ctx_set_timing(lst_ctx* ctx, int32_t enable);
/* After lst_ctx_sync with timing on: ms[i] = duration of kernel i; returns the number of kernels
 * (<= cap) or a negative status.  names (may be NULL) receives static strings. */
int lst_ctx_kernel_times(lst_ctx* ctx, float* ms, const char** names, int32_t cap);

/* Number of kernel launches issued by the last lst_ctx_run. */
int lst_ctx_launch_count(lst_ctx* ctx);

/* Diagnostics of the last synchronised batch (after lst_ctx_sync).  LST_STAT_PT_QUEUE: (seed, T3 / T5)
 * candidates that reached the exact cut list of the seed linking (CUTS.md section 7) -- the accepted ones plus
 * those the approximate pre-filters could not decide.  Returns the value (>= 0) or a negative lst_status. */
enum { LST_STAT_PT_QUEUE = 0, LST_STAT_WORKSPACE_MB = 1 };
int64_t lst_ctx_stat(lst_ctx* ctx, int32_t which);

/* ---- audit of the approximate cut cascades ------------------------------------------------------ */

/* MD, LS and the seed linking decide most candidates with cheaper arithmetic than CUTS.md's (approximate
 * reciprocal square roots and divisions, bounding circles) inside error bands; only what falls inside a band is
 * given to the exact cuts.  lst_ctx_audit checks, on the batch the context has just run
 * (after lst_ctx_sync, before the next lst_ctx_run), that none of those decisions was wrong: it re-evaluates EVERY
 * candidate of the three stages with the exact cuts only -- all hit pairs of a module (CUTS.md 3), all MD pairs along
 * the connection map (4), all (seed, T3) and (seed, T5) pairs of an event (7) -- and compares, per stage, the
 * number of candidates, of accepted and of near-threshold candidates and a 64-bit order-independent hash of the
 * accepted candidates' identities with what the chain counted and stored.  Index 0 MD, 1 LS, 2 pT3, 3 pT5; a
 * stage that the stage mask switches off (or pT without seeds) stays 0.  mismatches = how many of those
 * comparisons differ: 0 means every pre-filter decision of the batch agreed with the exact cuts and hid no
 * near-threshold candidate.  A debugging call: allocates a few hundred bytes, synchronises the stream, takes
 * milliseconds; never used by lst_ctx_run.  rep: host.  Errors: LST_ERR_ARG (no synchronised batch), the
 * batch's own error, LST_ERR_CUDA. */
typedef struct lst_audit_report {
  int64_t candidates[4], accepted[4], near[4];                   /* by the exact cuts on every candidate */
  int64_t chain_candidates[4], chain_objects[4], chain_near[4];  /* what the chain counted and stored */
  uint64_t hash_exact[4], hash_chain[4];
  int64_t mismatches;
} lst_audit_report;
int lst_ctx_audit(lst_ctx* ctx, lst_audit_report* rep);

/* ---- slot offsets from per-owner counts, stand-alone ------------------------------------------- */

/* Every stage of the chain is "owner -> a variable number of accepted objects" (an MD owns its
 * Line Segments, a seed its pT3s / pT5s); an owner's objects are stored from slot
 *     offsets[i] = counts[0] + ... + counts[i-1],   i = 0 .. n,     offsets[n] = number of objects.
 * The chain computes this with a one-launch tile scan (tiles publish their totals in status words and look back
 * over their predecessors'), which needs scratch memory beyond input and output: one ticket and one 64-bit
 * status word per tile of 1024 counts.  The two calls below run that scan on caller-owned arrays.
 *   counts:  DEVICE, n int32 (not read for n == 0), 16-byte aligned, each >= 0, total < 2^31.
 *   offsets: DEVICE, n + 1 int32, caller-owned, must not overlap counts.
 *   cuda_stream: a cudaStream_t as void* (NULL = the legacy default stream).
 * Errors: LST_ERR_ARG (n < 0, NULL or misaligned pointer), LST_ERR_CUDA.
 *
 * lst_scan_counts takes its scratch from cudaMalloc, waits for the result and frees the scratch again. */
int lst_scan_counts(const int32_t* counts, int32_t n, int32_t* offsets, void* cuda_stream);

/* The same scan for callers that must not allocate device memory: a trigger or reconstruction framework that
 * owns all device memory and forbids cudaMalloc / cudaFree inside its event loop (both synchronise the whole
 * device and stall every other stream on it), or any code running where the CUDA runtime refuses allocations.
 * This call makes no cudaMalloc, cudaFree or other allocating call.  Its scratch is a fixed array inside the
 * library image (about 128 KB; every GPU the library is loaded on keeps it until the process exits), which
 * bounds the size: n > LST_SCAN_STATIC_MAX_N returns LST_ERR_LIMIT and touches nothing.
 *   - Asynchronous: enqueues one memset and one kernel on cuda_stream and returns; offsets are valid once the
 *     stream has reached that point.
 *   - The first call on each device looks up the array's device address (that device must be current, as for
 *     every call); make that first call before starting any stream capture on the device.
 *   - All calls on a device share the one array, which still holds what the previous call left: each call
 *     clears the part it uses, in stream order.  Two calls that can overlap on the GPU (different streams, no
 *     dependency between them) race on it and give wrong offsets; order them, or use lst_scan_counts. */
#define LST_SCAN_STATIC_MAX_N (1 << 24)
int lst_scan_counts_static(const int32_t* counts, int32_t n, int32_t* offsets, void* cuda_stream);

#ifdef __cplusplus
}
#endif
#endif /* LST_H */

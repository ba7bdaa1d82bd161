/*
 * lhcb.h -- C ABI of the B200-native LHCb HLT1 Seeding + Matching hot path.
 *
 * The three calls follow the paper's statement of the problem (PAPER.md = arxiv/paper_2606_14480):
 *   lhcb_geom_init  : detector description + tunables                      (Eq. 1-23, Tables 1-2)
 *   lhcb_seeding    : per event, SciFi hits -> T-track seeds               (section 3)
 *   lhcb_matching   : seeds x VELO tracks (+ UT hits) -> Long tracks       (section 4)
 *
 * Conventions
 *   - Units: mm, MeV/c, q/p in 1/MeV, slopes dimensionless.  All floating point is IEEE float32.
 *   - Every pointer inside lhcb_events_t / lhcb_seeds_t / lhcb_velo_t / lhcb_ut_t / lhcb_long_t is a
 *     DEVICE pointer owned by the caller (e.g. a torch tensor's data_ptr()).  The *_t descriptor
 *     structs themselves, lhcb_geom_t and lhcb_derived_t live in HOST memory.
 *   - lhcb_seeding / lhcb_matching only enqueue work on `cuda_stream` (a cudaStream_t passed as
 *     void*; NULL = legacy default stream).  They do not synchronise and do not allocate.
 *   - Outputs are fully overwritten by each call (counts and status are reset by the call).
 *   - Return value: LHCB_OK (0) or a negative lhcb_status code; lhcb_error_string() names it.
 *     Per-event capacity overflow is NOT a return-code error: it is reported in the `status` output
 *     words (LHCB_ST_* bits), and the affected event-half keeps the entries that fitted.
 *   - One GPU per context.  A context may be used from one host thread at a time.
 */
#ifndef LHCB_H_
#define LHCB_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define LHCB_N_SCIFI_LAYERS 12
#define LHCB_N_UT_LAYERS 4
#define LHCB_NO_HIT 0xFFFFFFFFu

typedef enum {
  LHCB_OK = 0,
  LHCB_ERR_BAD_ARGUMENT = -1,   /* NULL pointer, negative size, inconsistent capacities */
  LHCB_ERR_BAD_GEOMETRY = -2,   /* not 6 x-layers + 6 stereo layers, seed triple not on x-layers, ... */
  LHCB_ERR_CUDA = -3,           /* a CUDA runtime call failed (see lhcb_last_cuda_error) */
  LHCB_ERR_NOT_INITIALISED = -4,
  LHCB_ERR_CAPACITY = -5,       /* requested capacities do not fit shared memory of the device */
  LHCB_ERR_STATIC_SCRATCH = -6  /* lhcb_seeding_static: more than LHCB_STATIC_MAX_EVENTS events in the batch */
} lhcb_status;

/* bits of the per-half / per-event `status` output words */
#define LHCB_ST_TRIPLET_OVERFLOW 1u   /* more three-hit combinations than max_triplets_per_half, or more two-hit work items in one
                                         tile of T1 hits than 4*max_xz_cand_per_half */
#define LHCB_ST_CAND_OVERFLOW 2u      /* more x-z candidates (>= min_x_hits) than max_xz_cand_per_half */
#define LHCB_ST_SEED_OVERFLOW 4u      /* more seeds than max_seeds_per_half */
#define LHCB_ST_HITS_OVERFLOW 8u      /* event-half has more hits than max_hits_per_half, or one of its zones 1,024 or more: half skipped */
#define LHCB_ST_MATCH_OVERFLOW 16u    /* more chi2-accepted pairs than max_match_cand_per_event */
#define LHCB_ST_LONG_OVERFLOW 32u     /* more long tracks than max_long_per_event */
#define LHCB_ST_VELO_OVERFLOW 64u     /* more VELO tracks than max_velo_per_event: event skipped */
#define LHCB_ST_UT_OVERFLOW 128u      /* more than 65534 UT hits in one event: event skipped */
#define LHCB_ST_BAD_RAW_HIT 512u       /* lhcb_prepare: a raw hit with zone >= 24 or a non-finite x: event passed through unsorted */
#define LHCB_ST_UV_QUEUE_OVERFLOW 256u /* stereo stage: survivors or queued u/v combinations exceed the shared work region */

/* Detector description and tunables.  Host POD, copied by lhcb_geom_init.
 * Citations: PAPER.md line / equation; "A<n>" = reading listed in DESIGN.md. */
typedef struct {
  float scifi_z[LHCB_N_SCIFI_LAYERS];          /* layer z, ascending                               L33 */
  float scifi_tan_alpha[LHCB_N_SCIFI_LAYERS];  /* tan(stereo angle); exactly 0 for the six x-layers L33 */
  float z_ref, d_ratio;                        /* Eq. 1 (L69-72) */
  float p_min, inv_p_a, inv_p_b;               /* Eq. 5-8 (L114-131); a, b per MeV (A1) */
  float alpha0, alpha1;                        /* Eq. 9-10 (L137-143) */
  int32_t iter_layers[2][3];                   /* T1,T2,T3 x-layer of each iteration (L78, A5) */
  float kappa_cx;                              /* c_x = polarity*q*kappa/p  (A3) */
  float cx_band[4];                            /* third-hit band f_lo, f_hi, d_lo, d_hi (Fig. 6, A4) */
  float tol_x_ext, tol_uv;                     /* 1 mm (L90), 2 mm (L215) */
  int32_t min_x_hits, min_uv_hits;             /* 5 (L90; must be 5 or 6), 4 (A9) */
  int32_t uv_first_layer[2];                   /* first stereo layer of the two UV passes (L215, A9) */
  float sigma_hit, chi2x_max, chi2y_max;       /* chi2/ndf cuts (L90, A6) */
  float y_min, y_max, y_half_tol;              /* detector halves: y>0 / y<0 (L372) */
  float z_velo, z_scifi_state, z_match_y;      /* state planes; y matching plane at 10 m (L231) */
  float mag[5];                                /* A_x..E_x of Eq. 18, Table 1 (L255-261) */
  float gamma_ab[2];                           /* A_gamma, B_gamma of Eq. 20, Table 1 (L262-263) */
  float kick_pt;                               /* K_B: q/p = polarity*dtx/K_B (A10) */
  int32_t polarity;                            /* +1 / -1; used when no per-event polarity is given */
  float presel[4];                             /* |dx|,|dy|,|dtx|,|dty| of Eq. 21 (L281) */
  float match_tol[8];                          /* Eq. 23: 4/5, 10.12, 101.0, 1/5, 1.59, 212.1, tol_tx, 1/tol_ty */
  float chi2_match_max;                        /* 2 (L301) */
  float ut_z[LHCB_N_UT_LAYERS], ut_tan_alpha[LHCB_N_UT_LAYERS];   /* UTaX, UTaU, UTbV, UTbX (L315) */
  float ut_loose[LHCB_N_UT_LAYERS][4];         /* A, B [mm GeV], min, max per layer: Table 2 (L323-340) */
  float ut_tight[LHCB_N_UT_LAYERS][4];
  float ut_y_tol;                              /* strip y-coverage tolerance (O13) */
  float ut_strip_x0, ut_strip_pitch;           /* UT strip number s <-> x0 = ut_strip_x0 + s*ut_strip_pitch in float32 (lhcb_ut_t.strip; L315: 190 um pitch) */
  float ut_row_y0, ut_row_pitch;               /* UT strips come in sensor rows: row r covers y in [ut_row_y0 + r*ut_row_pitch,
                                                  that + ut_row_pitch] (lhcb_ut_t.row; BASELINE.json configs[1]: 14 rows of 100 mm) */
  int32_t min_ut_hits, ut_enabled;             /* 3 (L311); 0 disables the UT search (L307) */
  /* capacities; 0 selects the default in brackets */
  int32_t max_seeds_per_half;                  /* [256]  output slots per event-half */
  int32_t max_xz_cand_per_half;                /* [1024] fitted x-z candidates per event-half.  The same region first holds the work
                                                  items of the two-hit search: the T3 windows of one tile of T1 hits (one hit per
                                                  thread of the CTA), cut into runs of four T3 hits, may not number more than
                                                  4*max_xz_cand_per_half per iteration, else LHCB_ST_TRIPLET_OVERFLOW */
  int32_t max_long_per_event;                  /* [256]  output slots per event */
  int32_t max_hits_per_half;                   /* [6144] SciFi hits staged per event-half (<= 8000).  Whatever this value, a single
                                                  (half, layer) zone may hold at most 1,023 hits (zone-local indices are packed in
                                                  10 bits): a half with a larger zone is skipped with LHCB_ST_HITS_OVERFLOW */
  int32_t max_triplets_per_half;               /* [4096] three-hit combinations per half, both iterations together (the queue also takes the
                                                  room a half leaves unused below max_hits_per_half) */
  int32_t max_match_cand_per_event;            /* [384]  chi2-accepted seed-VELO pairs per event */
  int32_t max_velo_per_event;                  /* [512] */
  int32_t max_ut_per_event;                    /* [6144] UT hits staged in shared memory per event; events with
                                                  more are searched in global memory (slower, same result) */
} lhcb_geom_t;

/* Geometry-only constants the kernels use (O1).  Computed in double from the float
 * geometry and rounded once to float.  Exposed so that host logic can be tested without a GPU. */
typedef struct {
  int32_t xl[6], ul[6], slot_of_layer[LHCB_N_SCIFI_LAYERS];
  float zb[12], gz[12], tan_a[12], inv_tan[12], inv_z[12], zt[12];
  float ywin_a[2][12], ywin_b[2][12];
  int32_t l1[2], l2[2], l3[2];
  float dx3max[2], alpha_corr[2], r13[2], inv_dz13[2], z1[2], dz12[2], K[2], inv_K[2], G13[2];
  float a, b, kappa, inv_kappa, f_lo, f_hi, d_lo, d_hi, tol_x, tol_uv, chi2x_max, chi2y_max;
  float wx[7], wy[7];
  float zbS, gS, gpS;
  float zS, zV, dzyS, dzyV, mag[5], presel[4], cx0, cx1, cy0, cy1, inv_tol_tx, inv_tol_ty, chi2m_max;
  float inv_KB, Ag, Bg, inv_Bg, ut_dz[4], ut_dz2[4], ut_dz4[4], ut_tan[4], ut_y_tol;
  float ut_loose[4][4], ut_tight[4][4];
  float P[7][3][6];      /* x-z least-squares map per hit pattern (0: six hits, 1+k: x-slot k missing) */
  float Q[64][2][6];     /* y-z least-squares map per stereo-slot bitmask */
} lhcb_derived_t;

typedef struct lhcb_ctx lhcb_ctx;

/* SciFi hits of a batch of events (section 3; L372: tiled by detector half, sorted per layer). */
typedef struct {
  int32_t n_events;
  uint32_t n_hits;           /* length of hit_x */
  const uint32_t* zone_off;  /* [n_events*24+1]; zone = (event*2+half)*12+layer, half 0: y>0 */
  const float* hit_x;        /* [n_hits] ascending inside each zone; stereo layers: x at y=0 */
  const int8_t* polarity;    /* [n_events] +1/-1, or NULL -> geom.polarity */
} lhcb_events_t;

/* Raw SciFi hits of a batch of events, in any order inside each event: the input of lhcb_prepare. */
typedef struct {
  int32_t n_events;
  uint32_t n_hits;           /* length of x and zone */
  const uint32_t* off;       /* [n_events+1] first raw hit of each event */
  const float* x;            /* [n_hits] finite; stereo layers: x at y=0 */
  const uint8_t* zone;       /* [n_hits] half*12 + layer, in [0, 24); half 0: y>0 */
} lhcb_raw_t;

/* Seeds ("T tracks", L219).  Event-half h owns slots [h*max_seeds_per_half, +count[h]); the order
 * inside a slot range is unspecified.  cap_total = n_events*2*max_seeds_per_half. */
typedef struct {
  int32_t n_events;
  uint32_t* count;     /* [n_events*2] */
  float* state;        /* SoA [5][cap_total]: x, y, tx, ty, q/p at z_scifi_state */
  float* par;          /* SoA [7][cap_total]: ax, bx, cx, ay, by, chi2x, chi2y   (may be NULL for matching) */
  uint32_t* hits;      /* SoA [12][cap_total]: global hit index per layer or LHCB_NO_HIT (may be NULL for matching) */
  uint8_t* nx;         /* [cap_total] (may be NULL for matching) */
  uint8_t* nuv;        /* [cap_total] (may be NULL for matching) */
  uint32_t* status;    /* [n_events*2] LHCB_ST_* bits */
} lhcb_seeds_t;

/* VELO track states at z_velo (L239-244). */
typedef struct {
  int32_t n_events;
  const uint32_t* off;       /* [n_events+1] */
  const float *x, *y, *tx, *ty;
  const int8_t* polarity;    /* [n_events] or NULL -> geom.polarity */
} lhcb_velo_t;

/* UT hits (L305-342): per (event, layer) sorted by x0 = x at y=0; strip covers [y_lo, y_hi].  The y coverage
 * comes either as the sensor row of the strip (one byte per hit: y_lo = ut_row_y0 + row * ut_row_pitch and
 * y_hi = y_lo + ut_row_pitch, evaluated in float32; y_lo / y_hi may then be NULL) or, when row is NULL, as two
 * floats per hit.  Rows are staged in shared memory beside x0; the float form is read from global memory. */
typedef struct {
  uint32_t n_hits;           /* length of x0, y_lo, y_hi, row */
  const uint32_t* off;       /* [n_events*4+1] */
  const float *x0, *y_lo, *y_hi;
  const uint8_t* row;        /* [n_hits] or NULL */
  const uint16_t* strip;     /* [n_hits] or NULL: strip numbers, x0 = ut_strip_x0 + strip * ut_strip_pitch.  Read by
                                lhcb_reconstruct_host only, which then ships 2 bytes per hit instead of the 4 of x0 and
                                decodes on the device; lhcb_matching reads x0 */
} lhcb_ut_t;

/* Long tracks.  Event e owns slots [e*max_long_per_event, +count[e]); order unspecified.
 * cap_total = n_events*max_long_per_event. */
typedef struct {
  uint32_t* count;     /* [n_events] */
  uint32_t* seed_idx;  /* [cap_total] slot index into lhcb_seeds_t arrays */
  uint32_t* velo_idx;  /* [cap_total] index into lhcb_velo_t arrays */
  uint32_t* ut_idx;    /* SoA [4][cap_total] index into lhcb_ut_t arrays or LHCB_NO_HIT */
  uint8_t* n_ut;       /* [cap_total] */
  float* qop;          /* [cap_total] q/p: UT-refined (Eq. 20) if UT hits were added, else the kick estimate */
  float* chi2;         /* [cap_total] chi2_match of Eq. 22 */
  uint32_t* status;    /* [n_events] LHCB_ST_* bits */
  float* ghost;        /* [cap_total] ghost probability (L346); written only while a network is set
                          (lhcb_set_ghost_nn); may be NULL */
} lhcb_long_t;

/* Host only.  Fills `out` from `g` (no CUDA call).  Returns LHCB_OK or LHCB_ERR_BAD_GEOMETRY /
 * LHCB_ERR_BAD_ARGUMENT.  lhcb_geom_init uses exactly this function. */
int lhcb_geom_derive(const lhcb_geom_t* g, lhcb_derived_t* out);

/* Creates a context on CUDA device `device`: derives the constants, uploads the tables, checks the
 * shared-memory budget of the capacities.  *out is owned by the caller until lhcb_destroy. */
int lhcb_geom_init(const lhcb_geom_t* g, int device, lhcb_ctx** out);
void lhcb_destroy(lhcb_ctx* ctx);

/* The geometry the context holds, with capacity defaults resolved. */
int lhcb_get_geom(const lhcb_ctx* ctx, lhcb_geom_t* out);

/* Bytes of the optional device workspace of a batch (see lhcb_order).  The two kernels keep every
 * intermediate in shared memory and run without a workspace (pass NULL). */
size_t lhcb_workspace_bytes(const lhcb_ctx* ctx, int n_events, size_t n_scifi_hits);

/* Optional scheduling step (batches of about 1000 events): sorts the
 * event-halves by their number of SciFi hits and the events by their number of UT hits (VELO states if
 * ut == NULL), heaviest first, into `workspace` (device memory, lhcb_workspace_bytes(n_events) bytes).
 * lhcb_seeding / lhcb_matching called with THIS workspace for THE SAME batch start their CTAs in that order,
 * which shortens the last wave of a small batch (for batches above 3,072 events, a dozen waves or more, the call does
 * nothing and the workspace is ignored); the results are the same in the same slots.  When lhcb_matching is the
 * call that follows lhcb_seeding directly on this context, with the same workspace, stream and batch size, it
 * is also launched as a programmatic dependent of that Seeding grid: its CTAs may start while the last Seeding
 * wave drains and wait for per-half "seeds written" flags kept in the workspace (enqueue nothing of your own in
 * that stream between the two calls).  In every other case (given seeds, another call in between) the Matching is
 * an ordinary launch.  `velo` may be NULL: without `ut` as well the Matching order is then the identity, the
 * workspace stays valid for lhcb_matching.  A workspace that lhcb_order has not filled for the batch must not be
 * passed to the two calls.  Enqueues one small kernel; does not synchronise. */
int lhcb_order(lhcb_ctx* ctx, const lhcb_events_t* events, const lhcb_velo_t* velo, const lhcb_ut_t* ut,
               void* workspace, void* cuda_stream);

/* Event preparation, the step before the hot path (hits tiled by detector half and layer;
 * the searches of section 3 need them sorted in x).  Inside each event the raw hits are
 * ordered by (zone, x, raw index): a stable sort.  Outputs (device pointers, caller-owned, overwritten):
 *   zone_off [n_events*24+1]  prefix offsets; event e keeps the range [raw.off[e], raw.off[e+1])
 *   hit_x    [n_hits]         x in sorted order: with zone_off, the lhcb_events_t that lhcb_seeding reads
 *   perm     [n_hits] or NULL perm[k] = raw index of sorted hit k
 *   status   [n_events]       0, or LHCB_ST_HITS_OVERFLOW (more raw hits in the event than
 *                             2*max_hits_per_half or than 65535) / LHCB_ST_BAD_RAW_HIT; such an event is
 *                             passed through unsorted with all its hits in zone 0 (lhcb_seeding then finds
 *                             nothing in it): reported, never silent.
 * Enqueues one kernel on cuda_stream; does not synchronise or allocate. */
int lhcb_prepare(lhcb_ctx* ctx, const lhcb_raw_t* raw, uint32_t* zone_off, float* hit_x, uint32_t* perm,
                 uint32_t* status, void* cuda_stream);

/* UV seeding version: 0 = iterative over the hits of a first stereo layer (the paper's
 * default, and the default here), 1 = Hough clusters (reading A20): a one-dimensional Hough
 * transform in t_y over all six stereo layers with 64 bins per detector half, a layer voting once per bin;
 * clusters of two adjacent bins ranked by the number of voting layers; up to eight clusters, each cut into
 * four finer t_y hypotheses; per hypothesis the closest hit within tol_uv in every layer; fit and choice of
 * the best combination as in the iterative version.  Takes effect from the next lhcb_seeding call. */
int lhcb_set_uv_hough(lhcb_ctx* ctx, int on);

/* Final selection with the ghost-killing network (reading A14b).
 * nn: HOST array of LHCB_GHOST_NN_SIZE floats  mu[8], isig[8], W1[32][8], b1[32], W2[32], b2, cut, margin
 * for the inputs (z_match, dx, dy, dtx, dty, chi2_match, eta_VELO, nHits_SciFi), standardised as
 * (v - mu) * isig; hidden ReLU, output logistic = ghost probability.  lhcb_matching then keeps the
 * candidates with ghost probability < cut (0.8) and removes a track that shares its VELO or its SciFi
 * segment with another kept track whose ghost probability is lower by at least margin (0.05; must be > 0)
 * -- instead of the chi2 ranking (A14).  nHits_SciFi = nx + nuv of the seed (12 if those arrays are NULL).
 * nn == NULL switches back to the chi2 ranking.  Copied to the device by this call (synchronous). */
#define LHCB_GHOST_NN_SIZE 339
int lhcb_set_ghost_nn(lhcb_ctx* ctx, const float* nn);

/* Seeding: x-z two-/three-hit search, extension, fit, clone kill, u/v addition, y fit (section 3).
 * One CTA per event-half.  `out` arrays must have cap_total = n_events*2*max_seeds_per_half slots.
 * workspace: NULL, or the workspace lhcb_order filled for this batch. */
int lhcb_seeding(lhcb_ctx* ctx, const lhcb_events_t* events, lhcb_seeds_t* out, void* workspace,
                 void* cuda_stream);

/* Seeding in heaviest-first CTA order without a workspace and without any allocation: lhcb_order + lhcb_seeding
 * in one call, for the caller who has no device memory to give and may not ask the driver for any.
 *
 * Who that is.  The algorithms of the paper run inside a trigger application that reserves
 * its device memory once at start-up and then loops over batches on several streams at a time.  Inside that
 * loop cudaMalloc / cudaFree are off limits: either call waits until the whole device is idle, so one stream's
 * allocation would stall every other stream's batch.  The same holds for a process whose device memory has
 * already been handed in full to another allocator (a framework's caching pool): a cudaMalloc there simply
 * fails.  Such a caller can still use plain lhcb_seeding (it needs no workspace), but then loses the
 * heaviest-first CTA order that shortens the last wave of a batch of about 1,000 events: lhcb_order wants a
 * workspace the caller cannot provide.  This call keeps that workspace inside the library instead.
 *
 * How.  The order tables and per-half flags (20 bytes per event) sit in one array of
 * LHCB_STATIC_MAX_EVENTS * 20 = 61,440 bytes that is part of the library image: every GPU on which this
 * library's kernels are loaded holds its own copy from module load until the process exits, whether or not
 * this call is ever made.  The call makes no cudaMalloc, cudaFree or other allocating call; it enqueues
 * two kernels (order, seeding) on cuda_stream and does not synchronise.  (lhcb_geom_init, at set-up, does allocate
 * its three small constant tables, about 11 KB; it is this per-batch call that allocates nothing.)
 *
 * events / out: exactly as for lhcb_seeding -- device pointers owned by the caller, outputs fully overwritten,
 * same seeds in the same slots as lhcb_seeding gives with or without a workspace.
 *
 * Limits and rules.
 *   - events->n_events <= LHCB_STATIC_MAX_EVENTS (3,072), else LHCB_ERR_STATIC_SCRATCH is returned and nothing is
 *     launched; split the batch or use lhcb_order + lhcb_seeding with your own workspace.  (Above that size
 *     the heaviest-first order no longer pays and lhcb_seeding ignores a workspace anyway.)
 *   - The first call on a device looks up the array's device address (once per device, cached) before it
 *     launches anything; make that first call outside any stream capture, e.g. on a small warm-up batch.
 *   - All calls on one device share the one array, also across contexts and threads.  Each call rewrites every
 *     word its batch uses before reading it, so the previous call's contents never matter and calls that
 *     follow each other in one stream are safe.  Two calls that can run on the GPU at the same time
 *     (different streams, different contexts on the same device) race on the array and give undefined
 *     results: serialise them, or give all but one of them lhcb_order + a workspace of their own.
 *   - The array is private to this call: lhcb_matching afterwards takes workspace = NULL. */
#define LHCB_STATIC_MAX_EVENTS 3072
int lhcb_seeding_static(lhcb_ctx* ctx, const lhcb_events_t* events, lhcb_seeds_t* out, void* cuda_stream);

/* Matching: kink extrapolation, preselection, chi2_match, UT hit search, one-to-one selection
 * (section 4).  `ut` may be NULL (no UT in the data taking, L307).  Of the seeds, count and state are
 * read; nx / nuv if given and a ghost network is set; hits if given: two seeds with bit-identical states
 * (twins from duplicate hits at the same x) tie exactly in chi2_match, and the tie is decided by their hit
 * lists in lexicographic order (layer 0 first), without hit lists by the lower slot (reading A21),
 * so the set of long tracks does not depend on the order in which lhcb_seeding wrote the seeds. */
int lhcb_matching(lhcb_ctx* ctx, const lhcb_seeds_t* seeds, const lhcb_velo_t* velo, const lhcb_ut_t* ut,
                  lhcb_long_t* out, void* workspace /* NULL or lhcb_order's */, void* cuda_stream);

/* ---- host-buffer pipeline (end-to-end path: H2D copies + seeding + matching + compaction + D2H copies) ----
 * A pipeline owns device buffers sized at creation, three CUDA streams (copies in, kernels, copies out) and one
 * CUDA graph per slice of events.  lhcb_reconstruct_host takes lhcb_events_t / lhcb_velo_t / lhcb_ut_t with
 * HOST pointers (pinned memory for full copy/compute overlap; pageable memory works, slower; of lhcb_ut_t, row is
 * required, y_lo / y_hi are not read, and strip is shipped instead of x0 when given), splits the batch into slices, and overlaps the input copies of later
 * slices and the output copies of earlier ones with the kernels.  Per slice: lhcb_order, lhcb_seeding,
 * lhcb_matching and two compaction kernels that move seeds and long tracks from their fixed slots to dense
 * arrays, so that exactly the found entries are copied back.  It blocks until every output has landed.
 *
 * Outputs (HOST arrays owned by the caller, fully usable on their own):
 *   seeds ("T tracks", L219: "made available to other algorithms"): event-half h owns the dense entries
 *     [off[h], off[h+1]); the order inside a half is unspecified.
 *   long tracks: event e owns [off[e], off[e+1]); seed_idx is an index into the dense seed arrays above,
 *     velo_idx / ut_idx are indices into the caller's batch arrays.
 * `cap` = entries the caller's arrays can hold (row stride of the [k][cap] arrays); n = entries written.
 * Returns LHCB_ERR_CAPACITY if the batch exceeds the sizes given at creation or the dense arrays are too
 * small; on any error every stream is drained before returning. */
typedef struct {
  uint32_t cap, n;
  uint32_t* off;       /* [n_events*2+1] */
  float* state;        /* [5][cap]  x, y, tx, ty, q/p at z_scifi_state */
  uint16_t* hits;      /* [12][cap] per layer l: hit index relative to the first hit of the seed's (half, layer) zone, i.e.
                          global index = host_events.zone_off[half*12 + l] + hits[l], or 0xFFFF for no hit (half the bytes
                          of a global index on the way back) */
  uint8_t *nx, *nuv;   /* [cap] */
  float* par;          /* [7][cap] ax, bx, cx, ay, by, chi2x, chi2y, or NULL (not copied) */
  uint32_t* status;    /* [n_events*2] LHCB_ST_* bits */
} lhcb_host_seeds_t;
typedef struct {
  uint32_t cap, n;
  uint32_t* off;       /* [n_events+1] */
  uint32_t* seed_idx;  /* [cap] index into lhcb_host_seeds_t */
  uint32_t* velo_idx;  /* [cap] */
  uint32_t* ut_idx;    /* [4][cap] or LHCB_NO_HIT */
  uint8_t* n_ut;       /* [cap] */
  float *qop, *chi2;   /* [cap] */
  uint32_t* status;    /* [n_events] LHCB_ST_* bits */
} lhcb_host_long_t;
typedef struct lhcb_pipeline lhcb_pipeline;
/* max_seeds_total / max_long_total: entries of the device-side dense arrays (0: the slot capacity of the batch) */
int lhcb_pipeline_create(lhcb_ctx* ctx, int max_events, size_t max_scifi_hits, size_t max_velo, size_t max_ut_hits,
                         int slice_events, size_t max_seeds_total, size_t max_long_total, lhcb_pipeline** out);
void lhcb_pipeline_destroy(lhcb_pipeline* p);
int lhcb_reconstruct_host(lhcb_pipeline* p, const lhcb_events_t* host_events, const lhcb_velo_t* host_velo,
                          const lhcb_ut_t* host_ut, lhcb_host_seeds_t* seeds_out, lhcb_host_long_t* long_out);
/* bytes moved by the last lhcb_reconstruct_host call; returns the number of kernels it launched */
int lhcb_pipeline_last_bytes(const lhcb_pipeline* p, uint64_t* h2d, uint64_t* d2h);

const char* lhcb_error_string(int status);
/* cudaError_t of the last failing CUDA call made through this context (0 if none). */
int lhcb_last_cuda_error(const lhcb_ctx* ctx);
/* Number of kernels the last lhcb_seeding / lhcb_matching call launched. */
int lhcb_last_launch_count(const lhcb_ctx* ctx);
/* Launch configuration the capacities of this context select: out[0] threads per
 * seeding CTA, out[1] its dynamic shared memory in bytes, out[2] threads per matching CTA, out[3] its
 * dynamic shared memory.  Smaller capacities let more CTAs share an SM (L382: occupancy). */
int lhcb_launch_config(const lhcb_ctx* ctx, int out[4]);

#ifdef __cplusplus
}
#endif
#endif /* LHCB_H_ */

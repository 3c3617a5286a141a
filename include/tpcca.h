/* =========================================================================================
 * tpcca.h -- C-ABI boundary of the B200-native TPC sector cellular-automaton (CA) tracker.
 *
 * What the library computes: the hot path PAPER.md:21 (section 1, "the EPNs perform full online
 * track reconstruction of the TPC data. This is the most computing-intense part of the
 * synchronous processing ... The full TPC processing happens on the GPUs") names and
 * BASELINE.json:5 (north_star) fixes as five stages, defined step by step in DESIGN.md
 * section 3 (= SURVEY.md section 8(c)):
 *   S1 per-row y/z grid binning of clusters
 *   S2 neighbour finder: best up/down link pair
 *   S3 mutual-link confirmation ("link cleaner")
 *   S4 start-hit selection, ordered compaction
 *   S5 tracklet construction + fp32 Kalman helix fit   (Bz = 0.5 T)
 * and, beyond the five (SURVEY.md 8(f) "next" rows):
 *   S6 tracklet selector: per-cluster ownership, clone removal
 *   S7 track-residual front end of a track-model cluster compression
 *   S8 cross-sector merging of the selected tracks + Kalman refit of the merged chains
 * "clusters per sector and pad row in, links and fitted tracks out" (BASELINE.json:5).
 *
 * Every stage runs in hand-written CUDA kernels for sm_100a; there is NO CPU fallback: every
 * entry point that needs the device fails with TPCCA_E_CUDA when no usable device exists.
 *
 * Conventions
 *  - every call returns 0 (TPCCA_OK) or a negative code; no exceptions, no exit(), no stdout;
 *    tpcca_last_error(ctx) gives a human-readable message for the last failing call.
 *  - plain pointers and sizes only.  Each pointer argument says whether it is HOST or DEVICE.
 *  - a context is not thread-safe; use one context per host thread / per stream.
 *  - index space of all outputs: "sorted position" = position of a cluster inside its sector
 *    after S1 (ascending (row, bin, original index)); order[] maps sorted -> original index.
 *    All cluster indices stored in outputs are SECTOR-LOCAL sorted positions; -1 = none.
 *  - arithmetic: every + - * / sqrt is one IEEE-754 binary32 round-to-nearest operation, no
 *    FMA contraction, no flush-to-zero; inputs containing NaN/Inf are
 *    undefined behaviour.
 * ========================================================================================= */
#ifndef TPCCA_H_
#define TPCCA_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define TPCCA_OK            0
#define TPCCA_E_ARG        -1   /* NULL / out-of-range argument                                  */
#define TPCCA_E_STATE      -2   /* wrong call order (e.g. run before all sectors were loaded)   */
#define TPCCA_E_CUDA       -3   /* CUDA runtime error or no usable device (message has details) */
#define TPCCA_E_WORKSPACE  -4   /* caller's workspace too small, or a device-side capacity       */
                                /* (max_start_hits) overflowed: nothing is silently truncated   */
#define TPCCA_E_RANGE      -5   /* a cluster's row >= n_rows (detected on the device in S1)      */

#define TPCCA_MAX_ROWS     256  /* n_rows limit of this build (the ALICE TPC has 152)            */
#define TPCCA_MAX_SECTORS  64   /* n_sectors limit (the ALICE TPC has 36)                        */

#define TPCCA_MEM_HOST          0  /* pointer is HOST memory, the library copies                  */
#define TPCCA_MEM_DEVICE        1  /* pointer is DEVICE memory, the library copies (D2D)          */
#define TPCCA_MEM_DEVICE_BORROW 2  /* DEVICE memory, used in place; must stay valid until the     */
                                   /* next load of the same sector or destroy (load only)        */

#define TPCCA_STAGE_GRID       0x01u
#define TPCCA_STAGE_NEIGHBOURS 0x02u
#define TPCCA_STAGE_CLEAN      0x04u
#define TPCCA_STAGE_START      0x08u
#define TPCCA_STAGE_TRACKLETS  0x10u
#define TPCCA_STAGE_ALL        0x1Fu   /* the five stages of the hot path (BASELINE.json:5)             */
#define TPCCA_STAGE_SELECT     0x20u   /* S6 tracklet selector; needs S1-S5.  Limit: fewer than  */
                                       /* 2^23 = 8 388 608 tracklets per sector (the ownership key holds the track   */
                                       /* number in 23 bits); beyond, tpcca_sync reports TPCCA_E_WORKSPACE.  The 4e8  */
                                       /* cluster time frame has about 0.9 M per sector.                            */
#define TPCCA_STAGE_RESIDUALS  0x40u   /* S7 cluster residuals to the selected tracks; needs S1-S6 */
#define TPCCA_STAGE_MERGE      0x80u   /* S8 cross-sector merging + chain refit; needs S1-S7       */

/* which output groups tpcca_get_tracks delivers (HOST: copies) */
#define TPCCA_OUT_ORDER      0x01u  /* order                                      (S1)            */
#define TPCCA_OUT_GRID       0x02u  /* syz, bin_start, row_start                  (S1)            */
#define TPCCA_OUT_LINKS_RAW  0x04u  /* link_up_raw, link_dn_raw                   (S2)            */
#define TPCCA_OUT_LINKS      0x08u  /* link_up, link_dn                           (S3)            */
#define TPCCA_OUT_START      0x10u  /* start_hit                                  (S4)            */
#define TPCCA_OUT_TRACKS     0x20u  /* track table + hit CSR                      (S5)            */
#define TPCCA_OUT_ALL        0x3Fu
#define TPCCA_OUT_SELECTION  0x40u  /* owner, n_own, sel_track                    (S6)            */
#define TPCCA_OUT_TRACKS_SEL 0x80u  /* the track table + hit CSR of the SELECTED tracks only (S6): fills the S5    */
                                    /* fields of the view from the compact table (array lengths: n_selected and    */
                                    /* n_sel_hits instead of n_tracks and n_hits); not together with OUT_TRACKS   */
#define TPCCA_OUT_RESIDUALS  0x100u /* res (tpcca_residual records)                (S7)            */
#define TPCCA_OUT_MERGE      0x200u /* mg_* links and merged chains               (S8)            */

typedef struct tpcca_ctx tpcca_ctx;   /* opaque; owned by the library */

/* S7: one 16-byte record per cluster (sorted position): the selected track the cluster is attached to and its
 * residuals to that track's helix at the cluster's pad row. */
typedef struct {
  int32_t trk;            /* sector-local number of the SELECTED track owning the cluster; -1: none (stored raw)   */
  float   res_y, res_z;   /* y_c - y_track, (z_c - z_ref) - z_track; 0 if trk == -1                                */
  int16_t q_y, q_z;       /* rint(res * res_inv_quantum) (round half to even), clamped to +-32767                  */
} tpcca_residual;

/* Tracker tables (DESIGN.md 3 "Derived tables").  All table pointers are HOST arrays of length
 * n_rows, owned by the caller and copied by tpcca_create.  The tables are DATA: geometry, grid,
 * windows and cuts are never hard-coded in the kernels. */
typedef struct {
  int32_t n_sectors;               /* 1 .. TPCCA_MAX_SECTORS; sectors are independent units       */
  int32_t n_rows;                  /* 3 .. TPCCA_MAX_ROWS pad rows                                */
  const float   *row_x;            /* pad-row plane x [cm], strictly increasing                   */
  const float   *grid_y_lo;        /* S1: lower y edge of the grid of row r                       */
  const float   *grid_inv_bin_y;   /* S1: 1 / bin size in y                                       */
  const int32_t *grid_ny;          /* S1: number of y bins (>= 1)                                 */
  float          grid_z_lo;        /* S1: lower z edge (all rows)                                 */
  const float   *grid_inv_bin_z;   /* S1: 1 / bin size in z                                       */
  const int32_t *grid_nz;          /* S1: number of z bins (>= 1)                                 */
  const float   *nf_hy_up, *nf_hz_up;   /* S2: window half-widths towards row r+1                */
  const float   *nf_hy_dn, *nf_hz_dn;   /* S2: window half-widths towards row r-1                */
  const float   *nf_cut;           /* S2: upper cut on the best score                             */
  float kappa_per_qpt;             /* S5: d sin(phi)/dx = kappa_per_qpt * (q/pT); 0.2998e-3*Bz[kG] */
  float err2_y, err2_z;            /* S5: measurement variances                                   */
  float init_cov[5];               /* S5: diagonal of the reset covariance                        */
  float tc_win_y, tc_win_z;        /* S5: search window half-widths                               */
  float tc_gate;                   /* S5: chi2-like gate on dist2                                 */
  float max_sinphi;                /* S5: propagation fails beyond this |sin(phi)|                */
  float grid_margin;               /* S2/S5: safety margin when turning a window into a bin range */
  int32_t tc_max_gap;              /* S5: consecutive rows without a hit before stopping          */
  int32_t tc_min_hits;             /* S5: minimum hits of an emitted track                        */
  int32_t sel_max_shared_permille; /* S6: a tracklet is selected iff (n_hits - n_own) * 1000 <= this * n_hits     */
  float res_inv_quantum;           /* S7: residuals are quantised to rint(res * this), 16 bits (> 0)              */
  /* S8: sectors s, s' are neighbours iff s / sectors_per_side == s' / sectors_per_side and they are adjacent (cyclic)  */
  /* inside the side; no merging if sectors_per_side < 2 or n_sectors is not a multiple of it                           */
  int32_t sectors_per_side;        /* 18 for the ALICE TPC                                                        */
  float sector_cos, sector_sin;    /* cos / sin of the angle between neighbouring sectors (20 degrees)            */
  int32_t mg_max_row_gap;          /* the upper segment starts 1 .. this rows above the lower segment's last row  */
  float mg_dy, mg_dz, mg_dsin;     /* match windows at the upper segment's reference plane (> 0)                  */
  float mg_zpre;                   /* pre-cut on |z(upper at x_ref) - z(lower on its last row)| (> 0)             */
} tpcca_params;

/* Outputs of ONE sector.  With mem_space == TPCCA_MEM_DEVICE the pointers are DEVICE pointers
 * into the caller's workspace; with TPCCA_MEM_HOST they are HOST pointers to buffers owned by
 * the context (the library did the D2H copies).  Either way they stay valid until the next
 * tpcca_run / tpcca_load_clusters / tpcca_get_* (HOST) / tpcca_destroy on this context.
 * Arrays of stages that were not run are NULL with their counts 0. */
typedef struct {
  int64_t n_clusters;      /* clusters loaded for the sector                                     */
  int64_t n_bins;          /* grid bins of a sector = sum_r ny_r * nz_r                          */
  int64_t n_start;         /* S4 start hits                                                      */
  int64_t n_tracks;        /* S5 emitted tracks                                                  */
  int64_t n_hits;          /* S5 total hits of the emitted tracks                                */
  int64_t trk_stride;      /* elements between consecutive planes of par[] and cov[]             */
  /* S1 */
  const int32_t  *order;      /* [n_clusters] sorted position -> original index                  */
  const float    *syz;        /* [n_clusters][2] bin-sorted (y, z) pairs, interleaved            */
  const uint32_t *bin_start;  /* [n_bins + 1] first sorted position of each bin; last = n        */
  const int32_t  *row_start;  /* [n_rows + 1] first sorted position of each row                  */
  /* S2: raw links */
  const int32_t  *link_up_raw, *link_dn_raw;   /* [n_clusters]                                   */
  /* S3: reciprocal links */
  const int32_t  *link_up, *link_dn;           /* [n_clusters]                                   */
  /* S4 */
  const int32_t  *start_hit;  /* [n_start] ascending sorted positions                            */
  /* S5: tracks in start-hit order */
  const float    *x_ref;      /* [n_tracks] plane of the reference state                         */
  const float    *z_ref;      /* [n_tracks] z of the start hit; absolute z = z_ref + par[1]      */
  const float    *par;        /* par[i * trk_stride + t], i < 5: y, z_rel, sin(phi), dz/ds, q/pT */
  const float    *cov;        /* cov[k * trk_stride + t], k < 15: lower triangle, k = i(i+1)/2+j */
  const float    *chi2;       /* [n_tracks]                                                      */
  const int32_t  *n_hits_trk; /* [n_tracks] number of attached clusters                          */
  const int32_t  *n_fit;      /* [n_tracks] clusters used by the final (downward) fit            */
  const int32_t  *first_row, *last_row, *trk_start_hit;   /* [n_tracks]                          */
  const int32_t  *hit_offset; /* [n_tracks + 1] CSR offsets into hit_idx, hit_offset[0] = 0      */
  const int32_t  *hit_idx;    /* [n_hits] sorted positions, ascending row inside a track         */
  /* S6: tracklet selector */
  int64_t n_selected;         /* selected tracks of the sector                                   */
  int64_t n_sel_hits;         /* total hits of the selected tracks                               */
  const int32_t  *owner;      /* [n_clusters] track (sector-local number) owning the cluster; -1 */
  const int32_t  *n_own;      /* [n_tracks] hits of each S5 track that the track owns            */
  const int32_t  *sel_track;  /* [n_selected] ascending sector-local numbers of the selected     */
  /* S7: residual front end, per cluster (sorted position) */
  const tpcca_residual *res;  /* [n_clusters] one record per cluster                              */
  /* S8, per SELECTED track of the sector (n_selected entries each): the partner segment in a
   * neighbour sector above / below (sector, selected-track number there; -1 none), and -- for tracks that are the
   * lowest segment of a chain of >= 2 segments (mg_n_seg > 0) -- the Kalman refit over all hits of the chain,
   * expressed in the frame and relative to the z_ref of segment mg_frame_seg of the chain (0 = this track) */
  int64_t mg_stride;          /* elements between consecutive planes of mg_par / mg_cov          */
  const int32_t  *mg_next_sec, *mg_next_trk, *mg_prev_sec, *mg_prev_trk;
  const int32_t  *mg_n_seg, *mg_n_hits, *mg_n_fit, *mg_first_row, *mg_last_row, *mg_frame_seg;
  const float    *mg_x_ref, *mg_z_ref, *mg_chi2, *mg_par, *mg_cov;
} tpcca_tracks_view;

/* Bytes of DEVICE workspace that tpcca_create needs for at most `max_clusters_total` clusters
 * over all sectors and at most `max_start_hits` S4 start hits over all sectors
 * (max_start_hits <= 0: a default of max_clusters_total / 8 + 1024; the hard bound is
 * max_clusters_total / 2).  HOST call, no device needed.  Errors: TPCCA_E_ARG. */
int tpcca_workspace_bytes(const tpcca_params *params, int64_t max_clusters_total,
                          int64_t max_start_hits, size_t *out_bytes);

/* Create a context on CUDA device `cuda_device`.  `cuda_stream` is a cudaStream_t of that device
 * (NULL = the legacy default stream) on which every kernel and copy of this context is issued.
 * `workspace` is a DEVICE buffer of `workspace_bytes` bytes (256-byte aligned), owned by the
 * caller and used by the context until tpcca_destroy.  The capacities are the ones passed to
 * tpcca_workspace_bytes.  Errors: TPCCA_E_ARG (bad tables), TPCCA_E_CUDA (no device: there is no
 * CPU path), TPCCA_E_WORKSPACE (buffer too small; message names the required size). */
int tpcca_create(const tpcca_params *params, int cuda_device, void *cuda_stream,
                 void *workspace, size_t workspace_bytes,
                 int64_t max_clusters_total, int64_t max_start_hits, tpcca_ctx **out_ctx);

/* Hand the clusters of one sector to the context (BASELINE.json:5 "clusters per sector and pad
 * row in").  SoA arrays of length n: y, z fp32 local coordinates [cm], row = pad-row index.
 * x (= row_x[row]) and charge are part of the cluster record (BASELINE.json:7) but S1-S5 do not
 * read them: either may be NULL; when given they are only validated for nullness, never copied.
 * mem_space says where x, y, z, charge, row live (TPCCA_MEM_*).  Copies are asynchronous on the
 * context's stream; HOST arrays must stay valid until the stream has passed the copy (pinned
 * memory makes it truly asynchronous).  Sectors accumulate until tpcca_reset; sectors never
 * loaded are empty; loading a sector twice without a reset is TPCCA_E_STATE.  The sum of n over
 * sectors must not exceed max_clusters_total (TPCCA_E_WORKSPACE).  Loading invalidates the
 * outputs of earlier runs.  Errors: TPCCA_E_ARG, TPCCA_E_STATE, TPCCA_E_WORKSPACE, TPCCA_E_CUDA. */
int tpcca_load_clusters(tpcca_ctx *ctx, int sector, int64_t n, const float *x, const float *y,
                        const float *z, const float *charge, const uint16_t *row, int mem_space);

/* Start a new time frame: forget all loaded sectors and all outputs (no device work). */
int tpcca_reset(tpcca_ctx *ctx);

/* Run the stages in `stage_mask` (bit i = stage i+1; S6-S8: TPCCA_STAGE_SELECT, _RESIDUALS, _MERGE) over all sectors, asynchronously on the
 * context's stream.  A stage needs the outputs of the stages before it from this or an earlier
 * run on the same clusters (TPCCA_E_STATE otherwise).  Device-side failures (row out of range,
 * start-hit capacity overflow) are reported by the next tpcca_get_* / tpcca_sync call.
 * The tables of S6-S8 live in workspace regions that S1 / S5 use as scratch: a later run of S1 or S5 without S6 (S7,
 * S8) invalidates them (they are then reported as not run, never delivered stale).
 * Errors: TPCCA_E_STATE, TPCCA_E_CUDA (the message names the stage whose launch failed). */
int tpcca_run(tpcca_ctx *ctx, uint32_t stage_mask);

/* Wait for the stream and report device-side failures of the last run (TPCCA_E_RANGE,
 * TPCCA_E_WORKSPACE) or TPCCA_E_CUDA. */
int tpcca_sync(tpcca_ctx *ctx);

/* Outputs of one sector (BASELINE.json:5 "links and fitted tracks out").
 * mem_space: TPCCA_MEM_DEVICE (pointers into the workspace, no copy; synchronises the stream) or
 * TPCCA_MEM_HOST (asynchronous D2H copies on a copy stream owned by the context into a context-owned
 * PINNED host arena, then one synchronise of that copy stream; par/cov are packed with trk_stride =
 * n_tracks).  `what` selects the output groups (TPCCA_OUT_*); groups not selected, or whose stage was not
 * run, are NULL.  A HOST call waits only for the last stage whose outputs it asks for: asking for
 * ORDER | LINKS | START while S5 of the same tpcca_run is still running copies them concurrently with S5
 * (n_tracks / n_hits are then reported as 0; ask for TPCCA_OUT_TRACKS afterwards).  The other counts are
 * always filled.  Errors: TPCCA_E_ARG, TPCCA_E_STATE (nothing was run), plus those of tpcca_sync. */
int tpcca_get_tracks(tpcca_ctx *ctx, int sector, int mem_space, uint32_t what, tpcca_tracks_view *out);

/* The outputs of ALL sectors in one call: views[s] for s = 0 .. n_sectors - 1, otherwise as tpcca_get_tracks.  HOST:
 * every array of every sector lands in ONE pinned arena behind one synchronise of the copy stream (valid until the
 * next tpcca_get_* (HOST) call on this context). */
int tpcca_get_tracks_all(tpcca_ctx *ctx, int mem_space, uint32_t what, tpcca_tracks_view *views);

/* Totals over all sectors after a run: out[0..6] = n_clusters, n_start, n_tracks, n_hits,
 * n_bins (per sector), n_selected, n_sel_hits (S6; 0 if not run).  Synchronises the stream.
 * Errors as tpcca_sync. */
int tpcca_get_counts(tpcca_ctx *ctx, int64_t out[7]);

/* Device time of each stage [ms] of the run `runs_back` runs ago (0 = the last tpcca_run; the
 * context keeps the events of its last 16 runs), from CUDA events recorded on the context's
 * stream around the stages; ms[0..4] = S1..S5, ms[5] = S1..S5 together, ms[6] = S6, ms[7] = S7, ms[8] = S8.  A stage
 * that was not in that run's stage_mask reports exactly 0 (ms[5] spans whichever of S1..S5 ran).
 * Synchronises the stream.
 * Errors: TPCCA_E_ARG (runs_back outside 0..15), TPCCA_E_STATE (no such run). */
int tpcca_get_timings(tpcca_ctx *ctx, int runs_back, float ms[9]);

/* Work counters of the last run's S5 kernel, for the ALU roofline:
 * out[0] = Kalman propagations that moved the state, out[1] = Kalman updates,
 * out[2] = gate evaluations (phase A), out[3] = searches, out[4] = search candidates scored.
 * Synchronises the stream. */
int tpcca_get_work_counters(tpcca_ctx *ctx, int64_t out[5]);

/* Number of kernels the last tpcca_run launched (for bench.py's "gpu_launches"). */
int tpcca_get_launch_count(const tpcca_ctx *ctx, int64_t *out);

/* How the context was configured by tpcca_create from its capacities (for tests and logs): out[0] = log2 of the
 * z slices per S1 coarse bucket, out[1] = S1 coarse buckets per sector, out[2] = S2 kernel variant (hit-list
 * depth per side), out[3] = SMs of the device, out[4] = resident S2 blocks per SM, out[5] = max_clusters_total,
 * out[6] = max_start_hits, out[7] = workspace bytes in use.  No device work.  Errors: TPCCA_E_ARG. */
int tpcca_get_info(const tpcca_ctx *ctx, int64_t out[8]);

/* Message of the last failing call on this context ("" if none).  Never NULL.  With ctx == NULL:
 * the message of the last failing tpcca_create / tpcca_workspace_bytes of this thread. */
const char *tpcca_last_error(const tpcca_ctx *ctx);

/* Release the context (not the workspace, not borrowed inputs).  NULL is allowed. */
void tpcca_destroy(tpcca_ctx *ctx);

/* ---- time-frame streaming: sector-group pipeline --------------------------------
 * A pipeline owns n_groups contexts; group g handles the sectors [g * n_sectors / n_groups, (g + 1) * n_sectors /
 * n_groups) of every time frame on its own stream and its own host thread: H2D load, tpcca_run, D2H delivery.
 * Sectors are independent units (no halo, no exchange), so the copies of one group overlap the kernels of the
 * others, the first tracks are on the host after 1 / n_groups of the work, and one workspace holds 1 / n_groups of
 * the time frame. */
typedef struct tpcca_pipeline tpcca_pipeline;

/* Bytes of DEVICE workspace EACH group needs for at most max_clusters_group clusters / max_start_hits_group start
 * hits in one group (tpcca_workspace_bytes for the largest group).  HOST call.  Errors: TPCCA_E_ARG. */
int tpcca_pipeline_workspace_bytes(const tpcca_params *params, int n_groups, int64_t max_clusters_group,
                                   int64_t max_start_hits_group, size_t *out_bytes);

/* cuda_streams[g] (n_groups pairwise distinct cudaStream_t of cuda_device; TPCCA_E_ARG if any two are equal) and
 * workspaces[g] (DEVICE, 256-byte aligned, workspace_bytes_each bytes) are owned by the caller until
 * tpcca_pipeline_destroy.  Errors as tpcca_create. */
int tpcca_pipeline_create(const tpcca_params *params, int cuda_device, int n_groups, void *const *cuda_streams,
                          void *const *workspaces, size_t workspace_bytes_each, int64_t max_clusters_group,
                          int64_t max_start_hits_group, tpcca_pipeline **out);

/* One time frame through the pipeline.  n[s], y[s], z[s], row[s]: the clusters of sector s (arrays of n_sectors
 * entries; HOST -- pinned memory lets the copies overlap -- or DEVICE per mem_space; they must stay valid until the
 * call returns; DEVICE arrays are copied on the groups' streams, which know nothing of the stream that produced them:
 * the producer must have finished, or every group stream must be made to wait for it (cudaStreamWaitEvent), before
 * the call -- the Python binding does the latter with torch's current stream).  stage_mask / what as for tpcca_run /
 * tpcca_get_tracks, EXCEPT cross-sector merging: the groups are separate contexts that never see each other's tracks,
 * so TPCCA_STAGE_MERGE / TPCCA_OUT_MERGE are refused with TPCCA_E_ARG (run S8 on one context over all sectors).
 * views[s] (HOST array of n_sectors views) receives HOST pointers into the pinned arenas of the groups, valid until
 * the next run of this pipeline.  Blocks until every group has delivered.  Errors: those of tpcca_load_clusters / tpcca_run / tpcca_get_tracks of any group
 * (message names the group). */
int tpcca_pipeline_run(tpcca_pipeline *p, const int64_t *n, const float *const *y, const float *const *z,
                       const uint16_t *const *row, int mem_space, uint32_t stage_mask, uint32_t what,
                       tpcca_tracks_view *views);

/* Sector ranges of the groups (first_sector[n_groups + 1], may be NULL) and the host wall time [ms] each group's
 * thread spent in the last run (ms[n_groups], may be NULL).  Returns n_groups (or TPCCA_E_ARG). */
int tpcca_pipeline_get_groups(const tpcca_pipeline *p, int32_t *first_sector, float *ms);

/* Message of the last failing call (p == NULL: of the last failing create / workspace_bytes of this thread). */
const char *tpcca_pipeline_last_error(const tpcca_pipeline *p);

void tpcca_pipeline_destroy(tpcca_pipeline *p);

/* ---- S4 start-hit selection without any allocation (BASELINE.json:5 "start-hit selection") ------
 * For callers that cannot obtain device memory of their own at the moment of the call and hold no tpcca context:
 * a step of an online framework whose GPU memory was handed out once, in full, at start of run (a cudaMalloc there
 * has nothing left to take, and cudaMalloc / cudaFree stall all streams of the GPU while other time frames are being
 * processed); a plug-in living under a caching allocator (e.g. PyTorch's), which cannot see or reuse memory taken
 * behind its back; a monitoring hook that has the two link arrays of a sector and nothing else.  The regular path
 * (tpcca_create + tpcca_run) does not serve them: it needs a caller-allocated workspace and creates events, a copy
 * stream and pinned host buffers.
 *
 * This call creates and allocates NOTHING (no cudaMalloc / cudaFree / cudaMallocHost, no stream or event, no
 * allocating library routine).  The scratch the stage needs -- one count and one offset per 2048-cluster tile --
 * is a fixed 64 KiB array inside the library image; every GPU the library is used on holds those 64 KiB until the
 * process exits.  That fixes the limit: n_clusters <= TPCCA_NOALLOC_MAX_CLUSTERS (16 777 216, four config-3
 * sectors); a larger n_clusters is refused with TPCCA_E_ARG before anything is launched.
 *
 * Computes  start_hit = [ c ascending in [0, n_clusters) : link_dn[c] == -1 and link_up[c] >= 0 ]  on the CLEANED
 * links of ONE sector (the link_up / link_dn of tpcca_tracks_view, or the caller's own), i.e. exactly what stage S4
 * of tpcca_run writes.
 *   cuda_device, cuda_stream  device and cudaStream_t (NULL = default stream) the three kernels are queued on; the
 *                             call is asynchronous and leaves the caller's current device as it found it.
 *   link_up, link_dn          DEVICE, int32[n_clusters], read only (may be NULL when n_clusters == 0).
 *   start_hit                 DEVICE, int32[max_start_hits], output; slots >= *n_start are not written.
 *   n_start                   DEVICE, int32[1], output: the number of start hits FOUND.  If it exceeds
 *                             max_start_hits only the first max_start_hits were stored; the caller compares (the call
 *                             does not wait for the GPU, so it cannot report this itself).
 *   err_msg, err_msg_len      HOST buffer for the message of a failing call (may be NULL / 0); "" on success.
 * All arrays are the caller's and must stay valid until the stream has passed the call.
 *
 * The scratch is ONE array per GPU, shared by every call in the process, and keeps the numbers of the previous
 * call.  No part of it has to be zero on entry (each call overwrites what it later reads), so consecutive calls on
 * one stream, of any sizes, are independent.  Calls that can be on the same GPU at the same time -- two streams, or
 * two host threads with their own streams -- overwrite each other's counts and give wrong start hits: put them on one
 * stream or order them with events.
 *
 * The first call on a device does a one-time set-up: it asks the CUDA runtime for the device address of the scratch
 * (which makes the runtime load the library's code on that device if it has not yet).  Make that first call during
 * initialisation, outside any stream capture; later calls only queue three kernels.
 * Errors: TPCCA_E_ARG (negative or too large sizes, NULL pointers, cuda_device outside 0..63), TPCCA_E_CUDA (no
 * device -- there is no CPU path --, set-up or launch failure). */
#define TPCCA_NOALLOC_MAX_CLUSTERS 16777216
int tpcca_start_hits_noalloc(int cuda_device, void *cuda_stream, const int32_t *link_up, const int32_t *link_dn,
                             int64_t n_clusters, int32_t *start_hit, int64_t max_start_hits, int32_t *n_start,
                             char *err_msg, size_t err_msg_len);

/* Library version string, e.g. "tpcca 0.1 (sm_100a)". */
const char *tpcca_version(void);

#ifdef __cplusplus
}
#endif
#endif  /* TPCCA_H_ */

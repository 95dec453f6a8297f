/*
 * lst.h -- C-ABI of liblst.so: the data-parallel hot path of Line Segment Tracking
 * (arXiv 2207.08207) on one NVIDIA B200 (sm_100a).
 *
 *   hits -> mini-doublets (MD) -> segments (LS) -> triplets (T3) -> quintuplets (T5)
 *
 * The paper states the problem (PAPER.md:37 overview; :43 MD; :47-49 LS and module map;
 * :53 T3; :55 T5; :125 one kernel per object class, run in sequence; :143 no per-event
 * allocation; :147 several events in flight).  Every formula and constant is the frozen
 * reading in DESIGN.md section 1 ("SPEC").
 *
 * Conventions
 *  - Plain C linkage, plain pointers and sizes.  Every function returns an int status
 *    (LST_OK = 0, errors < 0); nothing throws, aborts or prints.
 *  - "host" / "device" is stated for every pointer.  Device pointers returned in views are
 *    owned by the library (they live in the context's arena, allocated once in lst_create)
 *    and stay valid until the next lst_load_event on the same slot or lst_destroy.
 *  - `cuda_stream` arguments are a cudaStream_t passed as void* (NULL = the legacy default
 *    stream).  lst_load_event / lst_run / lst_run_batch only ENQUEUE work (no host
 *    synchronisation, no allocation): they may be captured into a CUDA graph.
 *  - An event lives in a SLOT (0 .. n_slots-1).  Slots are independent: several may be in
 *    flight on different streams and distinct slots may be driven from distinct
 *    host threads.  One slot must not be used from two streams at once.
 *  - Object identity is by ORIGINAL hit index = position in the caller's hit arrays
 *    (reading 16).  Within a slot objects are numbered deterministically:
 *    MDs by (module, azimuth of the lower hit, azimuth of the upper hit; ties by original hit
 *    index), segments by (inner MD, outer MD), triplets by
 *    (first segment, second segment), quintuplets by (first triplet, second triplet).
 *  - Overflow of a per-slot capacity is never silent: lst_sync returns LST_ERR_OVERFLOW, the
 *    slot's outputs are invalid, lst_get_stats still reports the sizes that were needed.
 */
#ifndef LST_H_
#define LST_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define LST_N_LAYERS 6
#define LST_MAX_ROW 64

#if defined(__GNUC__)
#define LST_API __attribute__((visibility("default")))
#else
#define LST_API
#endif

enum {
  LST_OK = 0,
  LST_ERR_ARG = -1,      /* NULL / out-of-range argument, invalid geometry, map, module id or side */
  LST_ERR_CUDA = -2,     /* a CUDA runtime call failed (lst_last_cuda_error gives the code)        */
  LST_ERR_OVERFLOW = -3, /* a per-slot capacity was exceeded                                       */
  LST_ERR_STATE = -4,    /* call out of order (e.g. lst_get_* before lst_sync)                     */
  LST_ERR_NOMEM = -5,    /* arena allocation failed in lst_create                                  */
  LST_ERR_LIMIT = -6     /* size beyond the fixed maximum of the entry point that allocates nothing */
};

enum { LST_MD = 0, LST_SEG = 1, LST_T3 = 2, LST_T5 = 3,
       LST_CLEAN = 4, /* optional stage after LST_T5: duplicate cleaning of the quintuplets (lst_run_stage only) */
       LST_PIXEL = 5  /* optional stage after LST_T5 (with or without LST_CLEAN): pixel line segments -> pixel triplets and
                         pixel quintuplets (lst_load_seeds first; lst_run_stage only) */ };

typedef struct lst_ctx lst_ctx;

/* Detector description. HOST pointers, copied by lst_create; the caller keeps ownership.
 * `layer` enters the computation (cut constants are per layer).  `phi` does not change any
 * result: it is the reference direction against which the hits of a module are ordered in
 * azimuth, so that the search for partners can be restricted to a window (DESIGN.md section
 * 6); it must be finite.  The rest is optional and unused.
 * PAPER.md:29 (pT modules), BASELINE.json configs[0]. */
typedef struct {
  int32_t n_modules;
  const int8_t* layer;  /* [n_modules] 0 .. LST_N_LAYERS-1 */
  const int8_t* kind;   /* [n_modules] 0 = PS, 1 = 2S (may be NULL) */
  const float* cx;      /* [n_modules] module centre (may be NULL) */
  const float* cy;
  const float* cz;
  const float* phi;     /* [n_modules] azimuth of the module normal, radians (required) */
} lst_geometry;

/* Module map: CSR lookup table module -> connectable modules of the next layer.
 * HOST pointers, copied by lst_create.  layer[targets[k]] must equal layer[src] + 1; a row
 * is strictly ascending and holds at most LST_MAX_ROW targets. */
typedef struct {
  int32_t n_modules;
  const int32_t* row_offsets; /* [n_modules + 1], non-decreasing, row_offsets[0] = 0 */
  const int32_t* targets;     /* [row_offsets[n_modules]] */
} lst_module_map;

/* Cut constants (all fp32) and runtime sizes. */
typedef struct {
  float half_kappa_max;
  float z_lum;
  float md_cos_eps[LST_N_LAYERS];
  float md_sin_eps[LST_N_LAYERS];
  float md_dz_res[LST_N_LAYERS];
  float md_eps[LST_N_LAYERS];
  float seg_cos_eps;
  float seg_sin_eps;
  float seg_z0_max[LST_N_LAYERS - 1];
  float t3_kappa_max;
  float t3_chi2rz_max[LST_N_LAYERS - 2];
  float sigma_z2[LST_N_LAYERS];
  float inv_sigma_z2[LST_N_LAYERS];
  float t5_dkappa_max;
  float t5_chi2rz_max[LST_N_LAYERS - 4];
  float t5_chi2xy_max;
  float t5_sigma_xy2_scaled;
  float t5_kappa_max;
  /* [P] pixel line segments -> pixel triplets [0] / pixel quintuplets [1] (DESIGN.md section 1 [P]) */
  float pix_dkappa_max[2];
  float pix_inv_var_xy[LST_N_LAYERS];
  float pix_inv_var_rz[LST_N_LAYERS];
  float pix_chi2xy_max[2];
  float pix_chi2rz_max[2];
  /* runtime */
  int32_t device;     /* CUDA device ordinal */
  int32_t n_slots;    /* event slots in the arena (>= 1) */
  int32_t cap_hits;   /* per-slot capacities, in objects */
  int32_t cap_md;
  int32_t cap_seg;
  int32_t cap_t3;
  int32_t cap_t5;
  int32_t timing;     /* != 0: record CUDA events around every kernel (lst_get_stats.stage_ms /
                         kernel_ms; for a batch they are kept on its first slot) */
  int32_t store_half; /* != 0: reduced-precision object store ("exploring data types such as half precision
                         floats"; DESIGN.md section 1 [H]): the per-object OUTPUT floats that no later selection reads -- MD
                         (dphi, dphichange), LS (sinS, z0, dphi, dphichange), T3 chi2rz, T5 (kappa_in, kappa_out, kappa_fit,
                         chi2xy, chi2rz) -- are stored as IEEE binary16, rounded to nearest even from the fp32 value; all
                         arithmetic and everything a selection reads stay fp32, so the object sets do not change.  The views
                         then expose these arrays through their *_h members and the fetched float payloads are binary16 */
  int32_t t5_dup_min_shared; /* [D] D4: quintuplets sharing at least this many of their 10 original hits
                         are duplicates (7).  Accepted range 6 .. 10 (lst_create returns LST_ERR_ARG otherwise): the
                         stage finds partners through a common mini-doublet, which >= 6 common hits imply and
                         <= 5 do not */
  int32_t cap_seeds;  /* [P] per-slot capacities: pixel line segments (16 k), pixel triplets (64 k), pixel quintuplets (64 k) */
  int32_t cap_pt3;
  int32_t cap_pt5;
  int32_t launches_in_flight; /* hint, >= 0: how many batched launches (lst_run_batch / lst_run_stage on different streams) the
                         caller keeps running side by side.  0 .. 3 (default 0): every stage grid is sized for half of the
                         machine, good for any use.  >= 4: the grids are sized so that FOUR launches of a stage together fill a
                         whole number of residency waves (BASELINE.json configs[2], 4 streams x 16 events: +0.9 % events/s;
                         a launch that runs alone, or two streams of 32 events, are then 15-50 % slower).  Results do not
                         depend on it */
} lst_config;

/* Fills *cfg with the frozen SPEC constants, device 0, 4 slots and capacities that hold the
 * PU300-like stress event of BASELINE.json configs[3] with margin. */
LST_API int lst_default_config(lst_config* cfg);

/* Hit SoA of one event (BASELINE.json configs[1]: "fp32 SoA (x, y, z, module id, sensor side)").
 * All five arrays are HOST pointers (on_device = 0) or all five DEVICE pointers (on_device = 1).
 * Fastest host form ("packed"): the five arrays back to back in ONE pinned block, each starting on a
 * 256-byte boundary (y = x + A, z = x + 2A, module = x + 3A, side = x + 4A as byte addresses, A = 4 n
 * rounded up to 256): the event travels as one copy-engine transfer at link speed.  Other pinned
 * (page-locked) host arrays are read by the binning kernel itself over PCIe, once and coalesced;
 * pageable host arrays go through five cudaMemcpyAsync.  They are borrowed until the stream has passed
 * the work enqueued by lst_load_event.  side: 0 = lower sensor (the anchor), 1 = upper. */
typedef struct {
  int32_t n;
  const float* x;
  const float* y;
  const float* z;
  const int32_t* module;
  const uint8_t* side;
  int32_t on_device;
} lst_hits;

/* Pixel line segments of one event ("pixel-based seeds ... line segments"; DESIGN.md section 1 [P]): the inner
 * tracker's estimate of a prompt helix per seed, fp32 SoA.  kappa: signed curvature in 1/cm with the sign convention of the
 * triplet curvature (lst_t3_view.md_kappa); (cphi, sphi): direction of the momentum at the beam line (a unit vector; seeds
 * whose direction is not one are still evaluated exactly, only slower); z0: z at the beam line, cm; t: cot(theta) = dz per
 * unit of transverse arc length.  All five HOST pointers (on_device = 0; pinned arrays are read by the kernel over PCIe,
 * pageable ones copied first) or all five DEVICE pointers (on_device = 1); borrowed until the stream has passed the work
 * enqueued by lst_load_seeds. */
typedef struct {
  int32_t n;
  const float* kappa;
  const float* cphi;
  const float* sphi;
  const float* z0;
  const float* t;
  int32_t on_device;
} lst_seeds;

/* Views: DEVICE pointers into the slot's object store + the object count. */
typedef struct {
  int32_t n;
  const int32_t* hits;         /* [n][2] original index of (lower, upper) hit                 */
  const int32_t* module;       /* [n]                                                         */
  const float* anchor;         /* [n][4] x, y, z, r of the anchor (lower) hit, 16-B aligned   */
  const float* ur_sina;        /* [n][2] r of the upper hit, sinA                             */
  const float* dphi_dphichange;/* [n][2]  (NULL when lst_config.store_half)                   */
  const int32_t* module_start; /* [n_modules + 1] MDs of module m are [start[m], start[m+1])  */
  const uint16_t* dphi_dphichange_h; /* [n][2] binary16 (NULL unless lst_config.store_half)   */
} lst_md_view;

typedef struct {
  int32_t n;
  const int32_t* md;       /* [n][2] inner MD, outer MD                                        */
  const float* f;          /* [n][4] sinS, z0, dphi, dphichange (NULL when store_half)         */
  const int32_t* md_start; /* [n_md + 1] segments with inner MD i are [start[i], start[i+1])   */
  const uint16_t* f_h;     /* [n][4] the same as binary16 (NULL unless store_half)              */
} lst_seg_view;

typedef struct {
  int32_t n;
  const int32_t* md_kappa; /* [n][4] MD1, MD2, MD3, bit pattern of kappa (fp32)                 */
  const int32_t* seg;      /* [n][2] first segment, second segment                              */
  const float* chi2rz;     /* [n] (NULL when store_half)                                        */
  const int32_t* seg_start;/* [n_seg + 1] triplets with first segment a are [start[a], start[a+1]) */
  const uint16_t* chi2rz_h;/* [n] binary16 (NULL unless store_half)                             */
} lst_t3_view;

typedef struct {
  int32_t n;
  const int32_t* md;       /* [n][5] MD1 .. MD5                                                 */
  const int32_t* t3;       /* [n][2] inner triplet, outer triplet                               */
  const float* f;          /* [n][5] kappa_in, kappa_out, kappa_fit, chi2xy, chi2rz (NULL when store_half) */
  const int32_t* t3_start; /* [n_t3 + 1] quintuplets with inner triplet A are [start[A], start[A+1]) */
  const uint16_t* f_h;     /* [n][5] the same as binary16 (NULL unless store_half)              */
} lst_t5_view;

/* Result of the optional duplicate-cleaning stage (DESIGN.md section 1 [D]): the
 * quintuplets that no better quintuplet sharing >= t5_dup_min_shared original hits removes -- the T5-only
 * track-candidate list. */
typedef struct {
  int32_t n;            /* quintuplets kept                                                       */
  const int32_t* t5;    /* [n] their indices into lst_t5_view, ascending                          */
  const uint8_t* keep;  /* [n_t5] 1 = kept                                                        */
  const float* score;   /* [n_t5] chi2xy + chi2rz, the fp32 sum of the fp32 values (also when store_half)  */
} lst_tc_view;

/* Result of the optional stage LST_PIXEL for kind 0 (pixel triplets: seed + triplet whose first MD is on layer 0 or 1) or
 * kind 1 (pixel quintuplets: seed + quintuplet): every (outer object, seed) pair that passes rule P0-P3, ordered by
 * (outer object, seed index).  Always fp32 (also with lst_config.store_half). */
typedef struct {
  int32_t n;
  const int32_t* link;         /* [n][2] seed index (position in the caller's seed arrays), index of the outer object
                                  (into lst_t3_view for kind 0, lst_t5_view for kind 1)                              */
  const float* f;              /* [n][3] chi2xy, chi2rz, kappa_object - kappa_seed                                   */
  const int32_t* object_start; /* [n_objects + 1] links of outer object o are [start[o], start[o+1])                 */
} lst_pix_view;

typedef struct {
  int32_t n_hits;
  int64_t needed[4];     /* objects that passed per class (may exceed the capacity on overflow) */
  int64_t candidates[4]; /* size of the search space per stage: pairs the method defines as
                            candidates (hit pairs of a module; MD pairs on map-connected modules;
                            segment pairs sharing an MD; triplet pairs sharing an MD)            */
  int64_t evaluated[4];  /* pairs the selection was actually evaluated on (<= candidates: the MD
                            and segment stages only look inside an azimuth window that is a
                            superset of what the selection can accept)                           */
  int32_t overflow;      /* bit k set: capacity of class k exceeded                              */
  int32_t bad_hits;      /* hits dropped because module id / side was out of range               */
  float stage_ms[5];     /* a0 .. a4; zeros unless lst_config.timing                              */
  float kernel_ms[12];   /* [0..2] a0: count (+ bin offsets and the slot's fresh header, by its last block), scatter, order;
                            [3..6] the MD, LS, T3, T5 kernel; [7..10] the four steps of LST_CLEAN (prepare, count + offsets
                            scan, fill, mark + list); [11] unused */
  int64_t rewalks[4];    /* chunks of 32 owners whose objects exceeded the on-chip stash and were walked twice */
  int32_t n_kept;        /* quintuplets kept by LST_CLEAN (0 if the stage was not run)                         */
  /* [P], index 0 = pixel triplets, 1 = pixel quintuplets (zeros unless LST_PIXEL was run) */
  int32_t n_seeds;       /* seeds loaded by lst_load_seeds                                                      */
  int64_t pix_needed[2];     /* links that passed (may exceed the capacity: overflow bits 4, 5)                 */
  int64_t pix_candidates[2]; /* the method's search space: (outer objects starting on layer 0 or 1) x seeds     */
  int64_t pix_evaluated[2];  /* pairs inside the azimuth window of the object's first anchor, all of which went
                                through the selection                                                           */
  int64_t pix_rewalks[2];
  float pix_ms[3];       /* seed binning kernel, pixel-triplet kernel, pixel-quintuplet kernel (lst_config.timing) */
} lst_stats;

/* Validates geometry and map, uploads the per-module tables, allocates the arena (the library allocates
 * here and nowhere else: nothing is allocated or freed per event).  cfg = NULL means lst_default_config.
 * Errors: LST_ERR_ARG (with nothing allocated), LST_ERR_NOMEM, LST_ERR_CUDA. */
LST_API int lst_create(const lst_geometry* geom, const lst_module_map* map, const lst_config* cfg, lst_ctx** out);
LST_API int lst_destroy(lst_ctx* ctx);

/* Step a0 ("a kernel that deals with pre-processing the hits and loading them"):
 * copies the hits to the device if they are on the host, bins them by (side, module), orders
 * each bin by azimuth (ties by original index) and derives r.  Asynchronous on `cuda_stream`.
 * Hits with an invalid module id or side are dropped and reported (lst_sync -> LST_ERR_ARG).
 * lst_load_events loads hits[b] into slot first_slot + b for b < n_slots with ONE set of
 * launches per 16 events.
 * Errors: LST_ERR_ARG (bad slot, n < 0, NULL arrays), LST_ERR_OVERFLOW (n > cap_hits). */
LST_API int lst_load_event(lst_ctx* ctx, int slot, const lst_hits* hits, void* cuda_stream);
LST_API int lst_load_events(lst_ctx* ctx, int first_slot, int n_slots, const lst_hits* hits, void* cuda_stream);

/* [P] Loads the pixel line segments of slots first_slot .. first_slot+n_slots-1 (seeds[b] into slot first_slot + b) and
 * orders them for the search (one kernel per 16 events).  Call it AFTER lst_load_event(s) of the same slots, on the same
 * stream (loading hits resets the slot, its seeds included).  Asynchronous.  The ordering kernel is forked onto a stream of
 * the library's own (after the work already enqueued on `cuda_stream`) so that it runs beside the stage kernels; LST_PIXEL,
 * lst_sync* and the next lst_load_event(s) of the slot join it again -- inside a stream capture one of them has to follow in the
 * same capture.
 * Errors: LST_ERR_ARG, LST_ERR_STATE (slot not loaded), LST_ERR_OVERFLOW (n > cap_seeds). */
LST_API int lst_load_seeds(lst_ctx* ctx, int first_slot, int n_slots, const lst_seeds* seeds, void* cuda_stream);

/* Steps a1..a4 for one slot / for slots first_slot .. first_slot+n_slots-1 in ONE set of
 * launches (the batch index is a grid dimension).  Asynchronous; no host synchronisation. */
LST_API int lst_run(lst_ctx* ctx, int slot, void* cuda_stream);
LST_API int lst_run_batch(lst_ctx* ctx, int first_slot, int n_slots, void* cuda_stream);
/* One stage only (LST_MD .. LST_T5) of a slot range; lst_run_batch == the four in order.  A stage needs the
 * one before it (LST_ERR_STATE otherwise); after a partial run the views / fetches of the classes built so far
 * are valid (BASELINE.json configs[4] runs the mini-doublet and segment stages only).  LST_CLEAN (duplicate
 * cleaning of the quintuplets, DESIGN.md section 1 [D]) is not part of lst_run / lst_run_batch: run it with
 * lst_run_stage after LST_T5.  LST_PIXEL (DESIGN.md section 1 [P]) likewise: after LST_T5 and lst_load_seeds
 * (LST_ERR_STATE otherwise), independent of LST_CLEAN. */
LST_API int lst_run_stage(lst_ctx* ctx, int first_slot, int n_slots, int stage, void* cuda_stream);

/* Waits for `cuda_stream`, reads the slot's counters back and returns its status:
 * LST_OK, LST_ERR_OVERFLOW, LST_ERR_ARG (bad hits were dropped), LST_ERR_CUDA. */
LST_API int lst_sync(lst_ctx* ctx, int slot, void* cuda_stream);

/* lst_sync for slots first_slot .. first_slot+n_slots-1 that were enqueued on `cuda_stream`: ONE
 * strided device-to-host copy of their counters and ONE stream synchronisation.  Returns LST_OK, or
 * LST_ERR_OVERFLOW if any slot overflowed, else LST_ERR_ARG if any slot dropped bad hits (per-slot
 * detail: lst_get_stats). */
LST_API int lst_sync_batch(lst_ctx* ctx, int first_slot, int n_slots, void* cuda_stream);

/* Valid after a successful lst_sync of the slot; LST_ERR_STATE otherwise. */
LST_API int lst_get_mds(lst_ctx* ctx, int slot, lst_md_view* out);
LST_API int lst_get_segments(lst_ctx* ctx, int slot, lst_seg_view* out);
LST_API int lst_get_triplets(lst_ctx* ctx, int slot, lst_t3_view* out);
LST_API int lst_get_quintuplets(lst_ctx* ctx, int slot, lst_t5_view* out);
/* Valid after LST_CLEAN was run (lst_run_stage) and the slot synced. */
LST_API int lst_get_track_candidates(lst_ctx* ctx, int slot, lst_tc_view* out);
/* Valid after LST_PIXEL was run and the slot synced; kind 0 = pixel triplets, 1 = pixel quintuplets. */
LST_API int lst_get_pixel_links(lst_ctx* ctx, int slot, int kind, lst_pix_view* out);
/* The same to HOST memory: link_out[n][2] (seed, outer object), f_out[n][3]; either may be NULL.  LST_ERR_ARG if
 * cap < n (lst_get_stats.pix_needed).  Synchronises `cuda_stream`. */
LST_API int lst_fetch_pixel_links(lst_ctx* ctx, int slot, int kind, int32_t* link_out, float* f_out, int64_t cap, void* cuda_stream);
/* Indices (into the quintuplet arrays, ascending) of the kept quintuplets to HOST memory: out[n_kept];
 * LST_ERR_ARG if cap < n_kept.  Synchronises `cuda_stream`. */
LST_API int lst_fetch_kept(lst_ctx* ctx, int slot, int32_t* out, int64_t cap, void* cuda_stream);
/* Valid after any lst_sync of the slot (also after an overflow). */
LST_API int lst_get_stats(lst_ctx* ctx, int slot, lst_stats* out);

/* Original-hit-index tuples of every object of class `kind` of a synced slot, gathered on the
 * device and copied to HOST memory: out[n][2 | 4 | 6 | 10] (hits of MD1 lower, MD1 upper,
 * MD2 lower, ...).  Writes min(n, cap_objects) rows; returns LST_ERR_ARG if cap_objects < n.
 * Synchronises `cuda_stream`. */
LST_API int lst_fetch_hit_indices(lst_ctx* ctx, int slot, int kind, int32_t* out, int64_t cap_objects, void* cuda_stream);
/* Float payload of class `kind` to HOST memory: MD [n][4] sinA, dphi, dphichange, r_anchor;
 * LS [n][4] sinS, z0, dphi, dphichange; T3 [n][2] kappa, chi2rz; T5 [n][5] as lst_t5_view.f.
 * fp32 values, or -- with lst_config.store_half -- binary16 values in the same order ([n][k] uint16_t; columns that are kept
 * in fp32 for the selections, e.g. sinA or kappa, are rounded to nearest even on the way out). */
LST_API int lst_fetch_values(lst_ctx* ctx, int slot, int kind, void* out, int64_t cap_objects, void* cuda_stream);

/* Result download for a batch of slots in one call (the end-to-end path of a multi-event
 * pipeline): synchronises the slots if they are not yet (lst_sync_batch), then
 * for slot first_slot + b gathers the hit-index tuples of class `kind` (LST_MD .. LST_T5, or LST_CLEAN =
 * the quintuplets kept by the cleaning stage only, in the layout of LST_T5) on the device and enqueues
 * their copy to the HOST buffer idx_out[b] ([n][2|4|6|10] int32) and the copy of the float payload
 * (layout and element type as lst_fetch_values: fp32, or binary16 with lst_config.store_half) to val_out[b].  idx_out / val_out may be NULL, and so may single
 * entries (nothing is copied for them).  cap_objects[b] = rows available in slot b's buffers;
 * counts[b] (may be NULL) receives the object count.  One gather launch per table for the whole
 * batch.  Pinned (page-locked) host buffers are written by ONE kernel per 16 slots directly over PCIe
 * (coalesced, each byte once); pageable ones through the slot's scratch area and one cudaMemcpyAsync
 * per buffer.  wait != 0: returns after the copies have completed; wait == 0: the work is only
 * enqueued and the buffers are complete once `cuda_stream` has been synchronised by the caller.  Errors: LST_ERR_STATE (a slot not run), LST_ERR_OVERFLOW,
 * LST_ERR_ARG (a buffer too small: nothing is copied), LST_ERR_CUDA. */
LST_API int lst_fetch_batch(lst_ctx* ctx, int first_slot, int n_slots, int kind, int32_t* const* idx_out,
                            void* const* val_out, const int64_t* cap_objects, int32_t* counts, int wait,
                            void* cuda_stream);

/* ---- module-map builder: the step before the path (DESIGN.md section 1 [B]) ---------------- */
/* Per-module inputs, HOST pointers, binary64: azimuth of the module normal, normal distance of the module
 * mid-plane from the beam line, distance between the two sensors, half width in r-phi, z range. */
typedef struct {
  int32_t n_modules;
  const int8_t* layer;      /* [n_modules] 0 .. LST_N_LAYERS-1 */
  const double* phi;
  const double* rho;
  const double* gap;
  const double* half_width;
  const double* z_lo;
  const double* z_hi;
} lst_map_geometry;
typedef struct {
  double pt_min;   /* GeV  (0.8: the paper's threshold) */
  double b_tesla;  /* T    (3.8) */
  double z0_max;   /* cm   (15)  */
  double pad_phi;  /* rad  (0.01) */
  double pad_z;    /* cm   (1)   */
} lst_map_params;
LST_API int lst_default_map_params(lst_map_params* params);
/* Builds the module map on `device`: module B of the next layer is connected to A iff the closed-form envelope
 * of the pT >= pt_min helices from A's edges meets B (rule B1-B4).  row_offsets: HOST [n_modules + 1], always
 * written; targets: HOST [cap_targets], rows ascending; *n_targets = number of connections.  params = NULL means
 * lst_default_map_params.  kernel_ms (may be NULL): [2] durations of the count and the fill kernel.
 * Errors: LST_ERR_ARG; LST_ERR_OVERFLOW if cap_targets is too small (row_offsets and *n_targets are valid: call
 * again with a buffer of *n_targets entries); LST_ERR_NOMEM; LST_ERR_CUDA. */
LST_API int lst_build_module_map(const lst_map_geometry* geom, const lst_map_params* params, int device, int32_t* row_offsets,
                                 int32_t* targets, int64_t cap_targets, int64_t* n_targets, float* kernel_ms);

/* The same map for callers that cannot allocate device memory (under CUDA graph capture, in a serving loop, in a harness
 * that forbids cudaMalloc): ONE entry point that calls no cudaMalloc / cudaFree / allocating library routine, creates no
 * event and never synchronises.  Three kernels are enqueued on `cuda_stream` (row lengths, exclusive scan, rows) and the call
 * returns; the outputs are complete once the caller has synchronised that stream.
 *   geom            HOST struct whose seven array pointers are DEVICE pointers ([n_modules] each, as in lst_map_geometry).
 *                   The values are NOT validated (they are on the device): the preconditions of lst_build_module_map
 *                   (layer in 0 .. LST_N_LAYERS-1, rho - gap/2 > 0, half_width > 0, finite) are the caller's to keep; whatever
 *                   the values, nothing outside the outputs is written.
 *   row_offsets     DEVICE [n_modules + 1], always written; row_offsets[n_modules] = number of connections.
 *   targets         DEVICE [cap_targets], rows ascending.  If the map has more than cap_targets connections only the entries
 *                   at CSR positions < cap_targets are written (the caller compares row_offsets[n_modules] with cap_targets:
 *                   there is no host-side status for it, the call has returned long before).  May be NULL iff cap_targets = 0.
 * The per-module row lengths between the first and the second kernel live in a file-scope device array of
 * LST_MAP_STATIC_MAX_MODULES ints (128 KiB, held by every GPU that loads the library until the process exits): n_modules above
 * that is rejected with LST_ERR_LIMIT before anything is enqueued.  Every call on a device shares that array and it keeps the
 * last call's contents: each call overwrites the entries it reads before reading them (nothing has to start at zero), but two
 * calls that overlap on the GPU (different streams, or graphs replayed concurrently) RACE on it -- keep them on one stream or
 * order them with events.  The first call on a device looks the array's address up (cudaGetSymbolAddress: may load the
 * module, so make that call outside a capture); later calls only enqueue.
 * Errors: LST_ERR_ARG (NULL pointers, n_modules <= 0, bad parameters, cap_targets < 0), LST_ERR_LIMIT, LST_ERR_CUDA. */
#define LST_MAP_STATIC_MAX_MODULES 32768
LST_API int lst_build_module_map_static(const lst_map_geometry* geom, const lst_map_params* params, int device,
                                        int32_t* row_offsets, int32_t* targets, int64_t cap_targets, void* cuda_stream);

/* Overflow recovery (BASELINE.json configs[3] "candidate-buffer overflow handling"; PAPER.md:143 sizes its buffers from the
 * data too): after lst_sync* returned LST_ERR_OVERFLOW for `slot`, fills *out with the context's configuration in which every
 * capacity that was exceeded is replaced by what the slot needed (lst_get_stats) times 1.25, rounded up to a multiple of 1024;
 * capacities that sufficed are kept.  A stage that overflowed feeds the later stages a clamped input, so their needs are
 * lower bounds: create a context from *out, run the event again, and repeat while it still overflows (at most once per
 * object class).  Returns LST_OK (also when nothing overflowed: *out is then the current configuration), LST_ERR_STATE if the
 * slot was not synced, LST_ERR_ARG. */
LST_API int lst_grown_config(lst_ctx* ctx, int slot, lst_config* out);

/* Bytes of the arena (all slots) and of one slot. */
LST_API int lst_arena_bytes(lst_ctx* ctx, int64_t* total, int64_t* per_slot);
/* Kernels launched by this context so far (for bench.py's gpu_launches). */
LST_API int64_t lst_launch_count(lst_ctx* ctx);
LST_API int lst_last_cuda_error(lst_ctx* ctx);
LST_API const char* lst_strerror(int status);
LST_API const char* lst_version(void);

#ifdef __cplusplus
}
#endif
#endif /* LST_H_ */

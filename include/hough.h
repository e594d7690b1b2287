/* hough.h -- C ABI of libhough: batched Hough-transform track finding on one B200 (sm_100a).
 *
 * The hot path of arxiv 2511.02742 ("GPU-based track-finding for the J-PARC muon g-2/EDM experiment"):
 *
 *   vote      every hit (u, v) adds one entry per theta bin to a 2-D histogram over (theta, rho),
 *             rho = u cos(theta) + v sin(theta)                       PAPER.md L90-92 (Sec. 4, Eq. 4.1)
 *             theta in [0, 180 deg), rho binned over a fixed range      PAPER.md L106 (Sec. 5)
 *   peaks     "the bin with the highest number of entries", here every strict local maximum with
 *             at least `vote_threshold` entries; clusters are the 8-connected components of the
 *             thresholded histogram                                   PAPER.md L94, L106; keyword L29
 *   assign    "selecting the hits that align with the straight line formed by the identified
 *             (theta, rho)"
 *
 * The paper fills one histogram per 10 ns time window in the shared memory of one CUDA block
 * (PAPER.md L114-116); an "event" here is one such window's 2-D point set.  Bin indices are computed
 * in fixed-point integer arithmetic from cos/sin tables defined by formula, so
 * every output except the two fp32 line parameters is an exact integer result.
 *
 * Conventions
 *   - d_* pointers are caller-owned DEVICE memory, h_* pointers are caller-owned HOST memory.  The library
 *     never keeps them past the call's stream work.  `stream` is a cudaStream_t passed as void* (NULL = the
 *     legacy default stream).
 *   - hough_vote / hough_find_clusters / hough_assign_hits only enqueue work on `stream`: no host
 *     synchronisation, no allocation.  Calls on one plan must be issued on one stream at a time (the plan
 *     owns scratch memory that the kernels reuse).
 *   - Return value: HOUGH_OK (0) or a negative hough_status code.  Nothing throws or aborts across the ABI.
 *   - Data-dependent conditions are not errors: an event with more than K local maxima reports the
 *     untruncated count in n_found and writes only the first K records; invalid hits (non-finite, or
 *     |u| or |v| > coord_max) cast no votes and get label -1; an event longer than max_hits_per_event
 *     (HOUGH_STATUS_EVENT_TOO_LONG), with a negative or decreasing offset, or ending beyond the plan's max_hits
 *     (HOUGH_STATUS_BAD_OFFSETS: its hits would lie outside buffers of that capacity) is skipped -- no candidates,
 *     n_found 0, its hits never read -- and sets that bit in the plan's device status word (hough_plan_status).
 *   - Records, counts and labels that a call takes as INPUT are caller data: a record that names no bin of the plan's
 *     grid attracts no hit, a label beyond the event's kept records is ignored; neither is used as an index.
 */
#ifndef HOUGH_H_
#define HOUGH_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    HOUGH_OK = 0,
    HOUGH_EINVAL = -1,  /* null pointer, negative size, misaligned buffer, bad descriptor field            */
    HOUGH_ERANGE = -2,  /* grid / fixed-point parameters fail the int32 proof, or a size exceeds the plan  */
    HOUGH_ECUDA = -3,   /* a CUDA runtime call failed; see hough_last_cuda_error()                         */
    HOUGH_ENOMEM = -4   /* host or device allocation failed                                                */
} hough_status;

enum { HOUGH_I32 = 0, HOUGH_U16 = 1 };            /* count_dtype: element type of accumulators dumped by hough_vote */
enum { HOUGH_STATUS_EVENT_TOO_LONG = 1, HOUGH_STATUS_BAD_OFFSETS = 2,      /* bits of the device status word */
       HOUGH_STATUS_INTERNAL = 4 };   /* set only by the -DHOUGH_BOUNDS debug build: an index check inside a kernel failed */
/* hough_plan_desc_t.flags.  The first two change only WHICH kernel computes an event, never a result:
 *   HOUGH_FLAG_GENERAL_ONLY  every event goes through the general kernel (the shared-memory-only fast kernel is not used)
 *   HOUGH_FLAG_SMALL_LISTS   the fast kernel's per-event lists get their smallest capacities, so that ordinary events
 *                            overflow them and are handed to the general kernel (exercises that hand-over in tests) */
enum { HOUGH_FLAG_GENERAL_ONLY = 1, HOUGH_FLAG_SMALL_LISTS = 2,
/*   HOUGH_FLAG_THETA_WRAP    DOES change results (a variant; reading B9): the line (theta + pi, rho)
 *                            is the line (theta, -rho) (Eq. 4.1), so the theta rows close into a ring with a twist -- past the
 *                            last row comes row 0 with its rho bins in reverse order.  With this flag local maxima (S2) and clusters
 *                            (S3) see those neighbours too: bin (n_theta - 1, r) touches bins (0, n_rho - 1 - r + {-1, 0, 1}).  A
 *                            track near theta = 0 is then one cluster instead of one at either end of the theta axis.  Needs the
 *                            default theta window, rho_min = -rho_max and n_theta >= 3 (else HOUGH_EINVAL); every event goes through
 *                            the general kernel; hough_find_tracks_peeloff and hough_find_two_stage do not accept such a plan. */
       HOUGH_FLAG_THETA_WRAP = 4 };

typedef struct hough_plan hough_plan_t;           /* opaque; created and destroyed by the library */

/* The (theta, rho) grid, thresholds and capacities of one plan.
 * theta spans [0, pi) unless a window is given: bin t stands for theta_t = pi t / n_theta (left edge; "0 to 180 deg").
 * rho spans the half-open range [rho_min, rho_max) in n_rho equal bins (histogram semantics). */
typedef struct {
    int32_t n_theta, n_rho;       /* >= 1; n_theta * n_rho <= 2^22                                          */
    double rho_min, rho_max;      /* same length unit as the hits                                           */
    double coord_max;             /* a hit is valid iff finite and |u|, |v| <= coord_max                    */
    int32_t hit_frac_bits;        /* H: hits are rounded to multiples of 2^-H (ties to even); < 0 -> 6      */
    int32_t acc_frac_bits;        /* F: fraction bits of the fixed-point rho bin coordinate; < 0 -> largest
                                     F <= 24 that keeps every intermediate (votes and bin centres) in int32 */
    int32_t vote_threshold;       /* T >= 1: a bin is "on" iff its count >= T                               */
    double assign_window;         /* w >= 0, in rho units: a hit may join a candidate iff its distance to
                                     the candidate's bin-centre line is <= w                               */
    int32_t max_candidates;       /* K in [1, 4096]: records kept per event                                 */
    int32_t count_dtype;          /* HOUGH_I32 or HOUGH_U16                                                 */
    int32_t max_events;           /* capacity: events per call                                              */
    int64_t max_hits;             /* capacity: hits per call; the kernels never read u, v or labels at or beyond it */
    int32_t max_hits_per_event;   /* capacity: hits in one event (HOUGH_U16 needs <= 65535).  Size it to the
                                     workload: the fast kernel stages this many hits in shared memory, at the
                                     cost of its other per-event lists (events that overflow those are still
                                     correct, but recomputed by the slower general kernel)                  */
    int32_t flags;                /* 0 or HOUGH_FLAG_* bits                                                 */
    int32_t device;               /* CUDA device ordinal                                                    */
    double theta_min, theta_max;  /* theta window in radians, bin t stands for theta_min + (theta_max - theta_min)
                                     t / n_theta; both 0 -> the paper's [0, pi); a narrower window
                                     spends the theta bins where the tracks are (slopes within +-1: [pi/4, 3pi/4)) */
} hough_plan_desc_t;

/* One track candidate: a local maximum of the event's accumulator.  32 bytes, little endian. */
typedef struct {
    int32_t theta_bin, rho_bin;   /* the peak bin (t, r)                                                    */
    int32_t votes;                /* its count                                                              */
    int32_t cluster_root;         /* slot, in this event's list, of the best-ranked peak of its cluster     */
    int32_t cluster_nbins;        /* bins in the 8-connected cluster (count >= T) that contains the peak    */
    float theta, rho;             /* line parameters of the bin: theta_t, and the rho bin centre            */
    int32_t reserved;             /* 0                                                                      */
} hough_candidate_t;

/* Constants a plan derived from its descriptor; for tests and diagnostics. */
typedef struct {
    int32_t hit_frac_bits, acc_frac_bits;  /* H, F                                                          */
    int32_t rho_offset_q;                  /* O_q = llround(-rho_min 2^F / d_rho)                           */
    int32_t assign_window_q;               /* W_q = llround(w 2^F / d_rho)                                  */
    int32_t strip_rows, n_strips;          /* theta rows of one shared-memory tile; tiles per event         */
    int32_t counter_bytes;                 /* width of the shared-memory counters (2 or 4)                  */
    int32_t threads_per_cta, ctas_per_sm, n_ctas, smem_bytes_per_cta;
    int32_t n_sm;
    /* fast kernel (0 in all fields when the plan cannot use it): column groups per tile row, launch shape and the
     * per-event capacities beyond which an event is left to the general kernel */
    int32_t fast_groups, fast_threads, fast_ctas, fast_smem_bytes;
    int32_t fast_hits_cap, fast_on_cap, fast_peak_cap, fast_strip_list_cap;
} hough_plan_info_t;

/* Validate the descriptor, derive F, build the int32 cos/sin tables C_q[t] = llround(cos(theta_t) M),
 * S_q[t] = llround(sin(theta_t) M), M = 2^(F-H) / d_rho, upload them, allocate scratch.  *out is set only on success. */
int hough_plan_create(const hough_plan_desc_t* desc, hough_plan_t** out);

/* Frees everything the plan owns.  Synchronises the device.  NULL is allowed. */
int hough_plan_destroy(hough_plan_t* plan);

/* Histogram filling only (Eq. 4.1): the materialising / diagnostic path.
 *   d_u, d_v      [N] fp32 hit coordinates, structure of arrays, 16-byte aligned
 *   d_offsets     [n_events + 1] int64, event e owns hits [offsets[e], offsets[e+1]); offsets[0] >= 0
 *   d_acc         nullable; [n_events][n_theta][n_rho] of count_dtype, theta-major, fully overwritten
 *   d_digest      nullable; [n_events] uint64: sum over bins of count * splitmix64(t * n_rho + r) mod 2^64 */
int hough_vote(hough_plan_t* plan, const float* d_u, const float* d_v, const int64_t* d_offsets, int32_t n_events,
               void* d_acc, uint64_t* d_digest, void* stream);

/* Vote + peak/cluster finding, fused: the accumulator lives only in shared memory.
 *   d_cands       [n_events][K] records; event e gets min(n_found[e], K) records in rank order
 *                 (votes descending, then t * n_rho + r ascending); the rest of its row is left untouched
 *   d_n_found     [n_events] int32: number of local maxima >= T of the event, not truncated to K */
int hough_find_clusters(hough_plan_t* plan, const float* d_u, const float* d_v, const int64_t* d_offsets,
                        int32_t n_events, hough_candidate_t* d_cands, int32_t* d_n_found, void* stream);

/* Hit-to-candidate assignment: label[h] = slot of the kept candidate whose bin-centre line is
 * nearest to hit h (fixed-point residual at the candidate's theta), among those within the window; ties go to
 * the lower slot; -1 if none or if the hit is invalid.
 *   d_cands, d_n_found   as written by hough_find_clusters for the same events (16- and 4-byte aligned)
 *   d_labels             [N] int32, every element of the events' ranges is written (skipped events: untouched); may be NULL
 *                        only for a plan with max_hits = 0 */
int hough_assign_hits(hough_plan_t* plan, const float* d_u, const float* d_v, const int64_t* d_offsets,
                      int32_t n_events, const hough_candidate_t* d_cands, const int32_t* d_n_found,
                      int32_t* d_labels, void* stream);

/* ---- stages around the core (O9-O13) ---- */

/* Detector planes (vanes) along u, for the "found" criterion of PAPER.md L136 (Sec. 7: "a track is regarded as found if its
 * hits are reconstructed and clustered in continuous five vanes"): plane k sits at u = plane_origin + k plane_pitch; a hit
 * belongs to its nearest plane, floor((u - origin) / pitch + 1/2), evaluated on the fixed-point coordinate. */
typedef struct {
    double plane_origin, plane_pitch;   /* pitch > 0; pitch * 2^H must round to >= 1                               */
    int32_t n_planes;                   /* 1 .. 64                                                                  */
    int32_t min_run;                    /* consecutive planes with a hit that make a track "found"; <= 0 -> 5       */
    int32_t wrap;                       /* != 0: the planes form a ring (plane n_planes - 1 is next to plane 0)     */
    int32_t reserved;                   /* 0                                                                        */
} hough_plane_geometry_t;

enum { HOUGH_FIT_FOUND = 1, HOUGH_FIT_DEGENERATE = 2 };

/* Refit of one kept candidate from the hits labelled with its slot.  32 bytes, little endian. */
typedef struct {
    int32_t n_hits;                     /* hits assigned to the slot                                                */
    int32_t max_run;                    /* longest run of consecutive planes that hold such a hit                   */
    uint64_t plane_mask;                /* bit k set iff plane k holds one                                          */
    float slope, intercept;             /* least-squares line v = slope u + intercept through the fixed-point hits  */
    int32_t flags;                      /* HOUGH_FIT_FOUND: max_run >= min_run; HOUGH_FIT_DEGENERATE: fewer than two
                                           hits, or all hits at one u (no slope; slope = intercept = 0)             */
    int32_t reserved;                   /* 0                                                                        */
} hough_fit_t;

/* Straight-line refit of every kept candidate (the stand-in for the paper's seed fit, "the corresponding
 * RecoHits lying along it are used as seeds", L112-114) and the found criterion (L136).  The sums are exact 64-bit integers
 * of the fixed-point coordinates, so the result does not depend on the order of the hits.
 *   d_n_found, d_labels   as written by hough_find_clusters / hough_assign_hits for the same events
 *   d_fits                [n_events][K]; event e gets min(n_found[e], K) records, the rest of its row is left untouched
 * HOUGH_ERANGE if the plan's coord_max * 2^H exceeds 2^15 or its max_hits_per_event exceeds 65535 (the sums would overflow). */
int hough_refit_tracks(hough_plan_t* plan, const float* d_u, const float* d_v, const int64_t* d_offsets, int32_t n_events,
                       const int32_t* d_n_found, const int32_t* d_labels, const hough_plane_geometry_t* geometry,
                       hough_fit_t* d_fits, void* stream);

/* Variant: the paper's own peak rule, one track at a time.  PAPER.md L94, L106: "a peak-finding
 * algorithm identifies the bin with the highest number of entries ... track seeds are found by selecting the hits that align
 * with the straight line".  Per event, repeated up to K times: histogram of the remaining hits -> global maximum under the
 * order (count descending, t * n_rho + r ascending); stop if its count < T; its hits (distance to the bin-centre line within
 * the assignment window) get the track's number as label and leave the hit set; a maximum none of whose hits lies in the
 * window ends the search.  K times the work of hough_find_clusters: for comparison, not for throughput.
 *   d_cands    [n_events][K]: track s of event e in record s (cluster_root = s, cluster_nbins = 0)
 *   d_n_found  [n_events]: number of tracks of the event
 *   d_labels   [N]: track number of every hit, or -1 */
int hough_find_tracks_peeloff(hough_plan_t* plan, const float* d_u, const float* d_v, const int64_t* d_offsets,
                              int32_t n_events, hough_candidate_t* d_cands, int32_t* d_n_found, int32_t* d_labels,
                              void* stream);

/* Variant: the paper's two-stage histogram.  PAPER.md L124, Fig. 5: "we perform the Hough
 * transformation into two stages: a coarse-binning histogram followed by a fine-binning histogram ... staying within the GPU's
 * shared memory constraints".  Per event: a coarse histogram whose bins merge coarse_theta x coarse_rho bins of the plan's grid
 * (coarse row T votes at the fine theta row in its middle); its strict local maxima >= T, the best K of them; for each a fine
 * patch of the 3 x 3 coarse bins around it, filled exactly; the patch maximum is a candidate if it has >= T votes; duplicates
 * are merged, records ranked by (votes descending, t * n_rho + r ascending), cluster_root = slot, cluster_nbins = 0.  An
 * approximation of hough_find_clusters by design: a track whose coarse bin is not a coarse local maximum is missed.
 * HOUGH_ERANGE if the coarse histogram and its lists exceed 200 KB of shared memory (choose coarser factors).
 *   d_cands, d_n_found   as for hough_find_clusters (usable by hough_assign_hits / hough_refit_tracks) */
int hough_find_two_stage(hough_plan_t* plan, const float* d_u, const float* d_v, const int64_t* d_offsets, int32_t n_events,
                         int32_t coarse_theta, int32_t coarse_rho, hough_candidate_t* d_cands, int32_t* d_n_found, void* stream);

/* Front end: RecoHits (x, y, z, t) of a batch of fills -> one event per time window, in the (phi, z) plane.
 * "the reconstructed hit points are divided into overlapping time windows of 10 ns, with a sliding step of
 * 5 ns.  Within each time window, the spatial coordinates (x, y, z) of the hits are transformed into the (phi, z) space".
 * Window w of every fill covers t0 + w step <= t < t0 + w step + width (times rounded to 2^-8 ns, ties to even).  phi =
 * atan2(y, x) in degrees, [-180, 180], by a 20-step integer CORDIC on x, y rounded to 2^-6 mm with the angle table
 * llround(atan(2^-i) 180 / pi 2^16): identical bits on every machine, within 4e-4 degree of atan2 for radii >= 1 mm. */
typedef struct hough_frontend hough_frontend_t;
typedef struct {
    double t0, window_width, window_step;   /* ns; width, step > 0 (PAPER.md: 10 and 5)                            */
    int32_t windows_per_fill;               /* >= 1; event index of window w of fill f = f * windows_per_fill + w   */
    double xy_max;                          /* a hit is valid iff finite, |x|, |y| <= xy_max (<= 512), (x, y) != 0  */
    int32_t max_fills;                      /* capacity: fills per call                                             */
    int64_t max_hits;                       /* capacity: input hits per call                                        */
    int32_t device;
    int32_t reserved;                       /* 0                                                                    */
} hough_frontend_desc_t;

enum { HOUGH_STATUS_OUTPUT_TRUNCATED = 8 };   /* front-end status bit: the output arrays were too small             */

int hough_frontend_create(const hough_frontend_desc_t* desc, hough_frontend_t** out);
int hough_frontend_destroy(hough_frontend_t* fe);

/* Enqueues the slicing on `stream` (no host synchronisation).
 *   d_x, d_y, d_z, d_t   [n_hits] fp32 RecoHits (mm, ns), structure of arrays
 *   d_fill_offsets       [n_fills + 1] int64, non-decreasing, fill f owns hits [fill_offsets[f], fill_offsets[f+1]);
 *                        a fill whose range does not lie inside [0, n_hits] is skipped and HOUGH_STATUS_BAD_OFFSETS is set
 *   d_u, d_v             [capacity] fp32 out: phi (degrees) and z of the windows' hits, window after window; inside a window
 *                        the hits keep their input order
 *   d_src                [capacity] int32 out: index of the input hit each output hit came from
 *   d_offsets            [n_fills * windows_per_fill + 1] int64 out: event offsets for hough_vote / hough_find_clusters / ...
 *                        always complete, even if the hits did not fit (then HOUGH_STATUS_OUTPUT_TRUNCATED is set and
 *                        d_offsets[last] tells the capacity that is needed; at most ceil(width / step) * n_hits) */
int hough_frontend_slice(hough_frontend_t* fe, const float* d_x, const float* d_y, const float* d_z, const float* d_t,
                         const int64_t* d_fill_offsets, int32_t n_fills, int64_t n_hits, float* d_u, float* d_v,
                         int32_t* d_src, int64_t* d_offsets, int64_t capacity, void* stream);

/* Reads and clears the front end's device status word.  Synchronises `stream`. */
int hough_frontend_status(hough_frontend_t* fe, int32_t* out, void* stream);

/* ---- helpers beyond the five ---- */

/* hough_find_clusters + hough_assign_hits on HOST buffers (pinned memory makes the copies asynchronous): the batch is cut
 * into chunks of events; a chunk's hits are copied to the device while the previous chunk is computed and the one before
 * that is copied back (three internal streams), then the call synchronises.  h_offsets[0] must be 0, h_offsets must be
 * non-decreasing and h_offsets[n_events] the number of hits.  Any output pointer may be NULL (then it is not copied
 * back); records beyond min(n_found, K) of an event are zero on the first call and otherwise unspecified. */
int hough_run_host(hough_plan_t* plan, const float* h_u, const float* h_v, const int64_t* h_offsets,
                   int32_t n_events, hough_candidate_t* h_cands, int32_t* h_n_found, int32_t* h_labels);

/* The same with the number of chunks given (1 .. 32; 0 = automatic, about 24 M hits per chunk). */
int hough_run_host_chunked(hough_plan_t* plan, const float* h_u, const float* h_v, const int64_t* h_offsets,
                           int32_t n_events, hough_candidate_t* h_cands, int32_t* h_n_found, int32_t* h_labels,
                           int32_t n_chunks);

/* Derived constants; h_cos_q / h_sin_q are nullable host arrays of n_theta int32 that receive the tables. */
int hough_plan_query(const hough_plan_t* plan, hough_plan_info_t* info, int32_t* h_cos_q, int32_t* h_sin_q);

/* Reads and clears the device status word (HOUGH_STATUS_* bits).  Synchronises `stream`. */
int hough_plan_status(hough_plan_t* plan, int32_t* out, void* stream);

/* Number of kernels the library has launched through this plan since creation. */
int64_t hough_plan_launch_count(const hough_plan_t* plan);

/* Diagnostic: reads and clears 16 per-phase SM-cycle sums (summed over CTAs) that the event kernel keeps only when
 * the library is built with -DHOUGH_PHASE_TIMERS; all zeros otherwise.  h_out16[15] is always the number of events the
 * last hough_find_clusters call on this plan handed from the fast kernel to the general kernel.  h_out16[14] / [13] are the
 * number of failed index checks and the site code of the first one since the last call (always 0 unless the library is
 * the -DHOUGH_BOUNDS debug build).  Synchronises `stream`. */
int hough_plan_debug_counters(hough_plan_t* plan, uint64_t* h_out16, void* stream);

/* Measures the conflict-free shared-memory atomic-add rate of the device (the roofline denominator of the
 * vote kernel): every SM runs nothing but `red.shared.add.u32` with lane = bank (addresses fixed in registers) for
 * about `millis` ms.
 * *ops_per_s receives the rate over the whole chip, *sm_clock_mhz the SM clock seen meanwhile. */
int hough_measure_smem_atomic_peak(int32_t device, double millis, double* ops_per_s, double* sm_clock_mhz);

const char* hough_strerror(int status);
const char* hough_last_cuda_error(void);          /* text of the last failed CUDA call on this thread, or "" */
int hough_version(void);

#ifdef __cplusplus
}
#endif
#endif /* HOUGH_H_ */

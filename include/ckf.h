/* ckf.h — C ABI of the B200-native combinatorial-Kalman-filter (CKF) track-finding library.
 *
 * What the entry points compute is the operation of arxiv 2505.22822 §2: "track parameters
 * and their covariances are propagated based on the fourth order Runge-Kutta-Nystrom method and the Kalman
 * Filter is applied to measurements on intersected sensor modules to calculate a chi2 value [...]  If the
 * chi2 is small enough, the measurement is attached to the track to make a new branch for the propagation
 * to the next sensor module."  Seeds in, track patterns out; geometry and magnetic
 * field cross to the device once, measurements/seeds/results per event.  The concrete rules
 * (units, stepping, navigation, gate, branching, caps) are DESIGN.md §3, following SURVEY.md §8(c).
 *
 * Conventions
 *   - Units: mm, GeV, tesla, c = 1 (time in mm).  Bound parameters (loc0, loc1, phi, theta, q/p, t).
 *   - All structs are POD and passed by const pointer; no C++ types or exceptions cross the ABI.
 *   - Return value: 0 (CKF_OK) on success, negative CKF_E_* otherwise; ckf_last_error() gives the text of the
 *     calling thread's last failure.
 *   - Threads: several host threads may call ckf_find / ckf_find_host on one handle, each on its own stream
 *     (one host thread per event pipeline).  With more streams than n_streams a workspace is recycled:
 *     the later call waits on the host until the earlier one has finished enqueuing and is ordered on the device
 *     after its work.
 *   - Malformed input (a seed module id out of range, a module_offsets array that is not monotonic or points beyond
 *     n) never causes an out-of-bounds access: the seed stops, the slice is clamped, and CKF_STATUS_BAD_INPUT is set.
 *   - ckf_find is ASYNCHRONOUS on `cuda_stream` and never allocates: every workspace is reserved in
 *     ckf_create from the max_* capacities (PAPER.md:84, :102 blame in-pipeline allocation for the lack of
 *     stream scaling).  Capacity overflow is never silent: it sets a bit in *status.  (One opt-in exception: with
 *     CKF_GRAPH=1 in the environment of ckf_create, a ckf_find that repeats the previous call's arguments is captured
 *     into a CUDA graph and replayed from then on; capture and instantiation allocate inside the CUDA runtime.)
 *   - There is no CPU fallback: without a CUDA device ckf_create fails with CKF_E_CUDA.
 */
#ifndef CKF_H_
#define CKF_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define CKF_ABI_VERSION 11

/* return codes */
#define CKF_OK 0
#define CKF_E_ARG (-1)     /* null pointer, bad size, unsupported value              */
#define CKF_E_CUDA (-2)    /* a CUDA runtime call failed (text in ckf_last_error)    */
#define CKF_E_CAPACITY (-3) /* n_seeds / n_measurements exceed the handle's capacity  */

/* bits of *ckf_tracks.status (device int32, written by ckf_find) */
#define CKF_STATUS_TRACK_OVERFLOW 1  /* more candidates than max_tracks: the first max_tracks are kept       */
#define CKF_STATUS_ENTRY_OVERFLOW 2  /* meas_idx capacity max_track_entries exceeded: later tracks dropped   */
#define CKF_STATUS_LINK_OVERFLOW 4   /* max_links or max_tips_per_level exhausted: some branches were cut    */
#define CKF_STATUS_BAD_INPUT 8       /* a seed's module id was out of range (that seed yields nothing), or
                                        module_offsets was not a valid CSR over [0, n] (slices were clamped)  */

/* stop reasons reported per candidate */
#define CKF_STOP_EXIT 1         /* left the detector (past the last layer / beyond half-z everywhere) */
#define CKF_STOP_HOLES 2        /* more than max_holes surfaces without a compatible measurement      */
#define CKF_STOP_NOT_OUTGOING 3 /* not radially outgoing when a cylinder portal was targeted          */
#define CKF_STOP_STEP_LIMIT 4   /* more than max_rk_steps_per_surface RKN4 trials on one move         */
#define CKF_STOP_NUMERIC 5      /* non-finite value or theta outside (0, pi)                          */
#define CKF_STOP_LEVEL_LIMIT 6  /* max_levels surfaces visited                                        */

typedef struct ckf_handle ckf_handle; /* opaque; owns device geometry, field, workspaces */

/* Detector: per-layer phi/z grid of planar modules (north_star "geometry store").  HOST pointers, copied
 * during ckf_create.  Module id = module_offset[l] + i_phi * n_z[l] + i_z; the module's local frame is
 * (axis_u, axis_v), its normal axis_u x axis_v; loc0 runs along axis_u, loc1 along axis_v.  Within a layer
 * all modules share half_v (the z pitch used by the navigator is 2*half_v of the layer's first module) and
 * n_phi >= 3.
 * What the navigator ASSUMES of the grid (it finds the 3x3 neighbourhood of a portal point by binning, it does not
 * search): on a barrel layer, module (i_phi, i_z) is centred at azimuth 2 pi i_phi / n_phi and at
 * z = -layer_half_z + (i_z + 1/2) * 2 half_v, tangent to the cylinder of radius layer_r with its normal pointing
 * outward; modules of one phi column are coplanar; neighbouring columns may overlap in phi by less than one module.
 * A geometry that violates this gives wrong module choices, not errors. */
typedef struct {
  int32_t n_layers;
  const double* layer_r;        /* [n_layers] mm, increasing                         */
  const double* layer_half_z;   /* [n_layers] mm                                     */
  const int32_t* n_phi;         /* [n_layers]                                        */
  const int32_t* n_z;           /* [n_layers]                                        */
  const int32_t* module_offset; /* [n_layers + 1]                                    */
  int32_t n_modules;
  const double* center;         /* [n_modules][3] mm                                 */
  const double* axis_u;         /* [n_modules][3] unit                               */
  const double* axis_v;         /* [n_modules][3] unit                               */
  const double* half_u;         /* [n_modules] mm                                    */
  const double* half_v;         /* [n_modules] mm                                    */
  const double* x_over_x0;      /* [n_modules]; 0 = no material                      */
  /* Endcap discs ("barrel + endcaps").  Both NULL = barrel only.  Barrel layers
   * come first, by increasing radius, the disc layers follow in any order.  For a disc layer l: layer_half_z[l] = signed
   * z of its plane, layer_r_min[l] .. layer_r[l] its radial acceptance, n_z[l] = number of rings, module id =
   * module_offset[l] + i_phi * n_z[l] + i_ring, ring pitch = 2 * half_v of the layer's first module; its modules lie in
   * the plane with loc1 (axis_v) radial and the normal axis_u x axis_v pointing away from z = 0. */
  const int32_t* layer_kind;    /* [n_layers] 0 barrel cylinder, 1 disc              */
  const double* layer_r_min;    /* [n_layers] inner radius of a disc (barrel: unused) */
} ckf_geometry;

/* Magnetic field (north_star "magnetic-field store").  HOST pointers, copied during ckf_create.
 * kind 1: value(ix,iy,iz) sits at origin + i*spacing; read by trilinear interpolation (x, then y, then z);
 * outside the grid the edge cell extrapolates linearly. */
typedef struct {
  int32_t kind;        /* 0 uniform, 1 grid                            */
  double uniform_b[3]; /* tesla                                        */
  int32_t n[3];
  double origin[3];
  double spacing[3];
  const float* grid;   /* [n0][n1][n2][3] tesla, float32 always        */
} ckf_field;

typedef struct {
  int32_t precision;   /* 32 or 64: element type T of every `void*` array below and of the covariance algebra.
                          The trajectory (position, direction, bound parameter vector) is float64 in both. */
  double chi2_max;     /* gate: chi2 < chi2_max (strict), 2 dof                                           */
  int32_t max_branches_per_surface; /* k best (chi2, index) passers become branches; 1..32                */
  int32_t max_candidates_per_seed;  /* cap on leaves per seed (R10); 1..256                     */
  int32_t max_holes;                /* a branch stops when its hole count exceeds this                   */
  int32_t min_measurements;         /* a stopped branch is emitted iff it holds at least this many       */
  double rk_tolerance_mm;           /* RKN4 local error bound per step                                   */
  double surface_tolerance_mm;      /* landing: a straight closing step once |distance| <= this          */
  double h_max_mm;                  /* largest step                                                      */
  double particle_mass_gev;         /* muon hypothesis                                      */
  int32_t max_rk_steps_per_surface;
  int32_t max_levels;               /* <= 64                                                             */
  /* capacities: every workspace and the bounds of the output arrays */
  int32_t max_seeds;
  int32_t max_measurements;
  int32_t max_tracks;               /* capacity of the per-track output arrays                           */
  int32_t max_track_entries;        /* capacity of meas_idx / entry_chi2                                 */
  int32_t max_links;                /* candidate-link buffer entries; 0 = 48 * max_seeds                 */
  int32_t max_tips_per_level;       /* live branch tips of one level, whole event; 0 = 8 * max_seeds     */
  int32_t n_streams;                /* independent workspaces; concurrent ckf_find calls up to this many */
  int32_t max_events_per_find;      /* largest batch of events one ckf_find may carry; 0 = 1 (see ckf_measurements) */
  int32_t energy_loss;              /* 1: mean energy loss of the muon hypothesis (Bethe, silicon, DESIGN.md rule E) in every
                                       crossed module of x_over_x0 > 0: q/p changes on leaving the module and the
                                       covariance is transported with d(q/p)'/d(q/p).  0: none (BASELINE configs)     */
  int32_t field_gradient;           /* 1: the transport Jacobian carries the field-gradient terms of PAPER.md ref [18]
                                       (DESIGN.md rule J2', reading A13): the step map is differentiated stage by stage
                                       including dB/dr of the interpolated field, and D gains its two position columns.
                                       No effect in a uniform field.  0 (BASELINE configs): ref [17], gradient neglected  */
  int32_t bidirectional;            /* 1: tips that move radially INWARD are navigated too (DESIGN.md rules N3''): they cross the
                                       inner layers against the module normals, pass the beam line and leave through the far
                                       side.  0 (BASELINE configs, reading A7): outward only, such tips stop NOT_OUTGOING    */
  int32_t max_seed_doublets;        /* ckf_seed: capacity of its middle-top doublet lists; its workspace (48 B per measurement
                                       + 12 B per doublet) is reserved in ckf_create.  0 = no ckf_seed on this handle */
  int32_t max_fit_tracks;           /* ckf_fit: candidates fitted per pass; sizes the state store reserved in ckf_create
                                       (max_levels states x min(max_fit_tracks, max_tracks, 262144) candidates x
                                       (12 float64 + 69 T): 3 GB at 262,144 in fp32).  0 = no ckf_fit on this handle */
} ckf_config;

/* Measurements of one event: CSR by module id (north_star).  DEVICE pointers, caller-owned, read-only.
 * A measurement's index is its position in loc/var and is what ckf_tracks.meas_idx reports.
 *
 * Batch of events (n_events = B > 1, at most config.max_events_per_find).  Events are independent,
 * so B of them may share ONE ckf_find: the caller concatenates their measurements (event 0 first) and their seeds and
 * addresses modules by the VIRTUAL id  event * n_modules + module  -- in module_offsets, which then has
 * B * n_modules + 1 entries over the concatenated arrays, and in ckf_seeds.module_id.  The library treats the batch as
 * one event in B replicas of the detector: every level of the branch loop then runs over the tips of all B events
 * (the per-level cost of the level-synchronous loop is shared), and nothing else changes: meas_idx reports positions
 * in the concatenated arrays, seed_id positions in the concatenated seeds (so the candidates of event e are those
 * whose seed_id lies in its seed range, contiguous in the output), last_module the real module id.  Capacities
 * (max_seeds, max_measurements, max_tracks, ...) count the whole batch.  Results per event are identical to those
 * of B separate calls (tested). */
typedef struct {
  int32_t n;
  const int32_t* module_offsets; /* [n_events * n_modules + 1]; (virtual) module m owns [off[m], off[m+1]) */
  const void* loc;               /* T[n][2] local position (loc0, loc1) mm             */
  const void* var;               /* T[n][2] variances mm^2                             */
  int32_t n_events;              /* 0 or 1: one event; B > 1: a batch, see above       */
} ckf_measurements;

/* Seeds: bound parameters + covariance on a module.  DEVICE pointers, caller-owned, read-only. */
typedef struct {
  int32_t n;
  const int32_t* module_id; /* [n]  (virtual id event * n_modules + module in a batch)  */
  const void* params;       /* T[n][6]  loc0 loc1 phi theta q/p t                */
  const void* cov;          /* T[n][36] row-major, symmetric                     */
} ckf_seeds;

/* Track candidates.  DEVICE pointers, caller-owned, caller-sized from max_tracks / max_track_entries.
 * Order: by seed id; within a seed by the level at which the branch stopped, then by branch order
 * (children of an earlier parent first, within a parent by (chi2, index) rank).  Deterministic.
 * Not de-duplicated (ambiguity resolution is a later stage). */
typedef struct {
  int32_t* n_tracks;       /* [1] number of candidates written (<= max_tracks)                       */
  int32_t* status;         /* [1] CKF_STATUS_* bits                                                  */
  int32_t* track_offsets;  /* [max_tracks + 1] CSR into meas_idx / entry_chi2                        */
  int32_t* meas_idx;       /* [max_track_entries] measurement indices in visit order, holes omitted  */
  int32_t* seed_id;        /* [max_tracks]                                                           */
  int32_t* n_holes;        /* [max_tracks]                                                           */
  int32_t* last_module;    /* [max_tracks] module of the last measurement                            */
  int32_t* stop_reason;    /* [max_tracks] CKF_STOP_*                                                */
  void* params;            /* T[max_tracks][6]  filtered parameters at the last measurement */
  void* cov;               /* T[max_tracks][36] their covariance, row-major                          */
  void* chi2_sum;          /* T[max_tracks]                                                          */
  void* entry_chi2;        /* T[max_track_entries] predicted chi2 of each attached measurement       */
} ckf_tracks;

/* Work counters of the last ckf_find on a workspace (for roofline accounting). */
typedef struct {
  int64_t tips;         /* branch tips processed (sum over levels)             */
  int64_t visits;       /* surface visits (gate evaluations of a whole module)  */
  int64_t rk_trials;    /* RKN4 trial steps                                     */
  int64_t rk_accepted;  /* accepted RKN4 steps                                  */
  int64_t gate_tests;   /* chi2 evaluations the method defines: sum of visited slice lengths */
  int64_t updates;      /* Kalman updates                                       */
  int64_t links;        /* candidate links appended                             */
  int64_t iterations;   /* levels that held at least one tip                    */
  int64_t gate_tests_executed; /* chi2 evaluations actually run: entries inside the loc0 windows
                                  (the rest of each slice is excluded by chi2 >= r0^2/S00) */
} ckf_counters;

/* Uploads geometry and field (once, at the first event) and reserves all workspaces.
 * All pointers inside geometry/field are HOST.  *out receives the handle.  Fails with CKF_E_CUDA when no
 * CUDA device of compute capability 10.x is present. */
int ckf_create(const ckf_geometry* geometry, const ckf_field* field, const ckf_config* config, ckf_handle** out);

/* Runs CKF track finding for one event on `cuda_stream` (a cudaStream_t; NULL = default stream).
 * Asynchronous; all pointers in measurements/seeds/out are DEVICE pointers that must stay valid until the
 * stream reaches the end of the call's work.  Up to n_streams calls may be in flight on different streams;
 * further streams are ordered after the call that last used the recycled workspace (also when that call is still
 * being enqueued by another host thread). */
int ckf_find(ckf_handle* handle, const ckf_measurements* measurements, const ckf_seeds* seeds, ckf_tracks* out,
             void* cuda_stream);

/* Same work with HOST buffers: copies measurements and seeds host->device, runs ckf_find, copies the
 * candidates device->host, all on `cuda_stream` (PAPER.md:51 transfer policy; BASELINE config 4).  Buffers
 * should be pinned for the copies to be asynchronous.  Device staging buffers belong to the handle.
 * SYNCHRONOUS: when it returns, the stream has been synchronised and the output arrays are filled up to *n_tracks /
 * track_offsets[*n_tracks] (what lies beyond is unspecified: the copies are sized from a guess, the previous call's
 * result + 1/8, so that one synchronisation per call suffices; the host arrays need their full capacity). */
int ckf_find_host(ckf_handle* handle, const ckf_measurements* measurements, const ckf_seeds* seeds, ckf_tracks* out,
                  void* cuda_stream);

/* ---- Kalman-filter track fit + RTS smoother over candidates ----------
 * "The filtered track parameters at the first measurement ... are estimated only with one measurement hence
 * least accurate.  Therefore, a Kalman Filter-based fitting, which runs a smoothing algorithm called the
 * Rauch-Tung-Striebel (RTS) smoother, is applied additionally to the tracks".
 * Rules K1-K5 of DESIGN.md 3: the forward filter walks each candidate's own path (same navigation, RKN4,
 * Jacobian, material and update rules as ckf_find) using the listed measurements in order; every visited
 * module is a state; the RTS recursion then runs backward over the states in float64.
 * Results.  DEVICE pointers, caller-owned, sized from max_tracks / max_track_entries like ckf_tracks. */
typedef struct {
  int32_t* status;      /* [max_tracks] 0 = fitted; else CKF_STOP_* of the forward pass, or CKF_STOP_NUMERIC when a
                           predicted covariance was not positive definite.  A track that is not fitted has zeros
                           in every other array                                                              */
  int32_t* n_states;    /* [max_tracks] modules the forward pass visited                                      */
  void* chi2_sum;       /* T[max_tracks] forward chi2 sum (equals ckf_tracks.chi2_sum)                        */
  void* last_params;    /* T[max_tracks][6]  forward-filtered state at the last measurement (= ckf_tracks.params) */
  void* last_cov;       /* T[max_tracks][36]                                                                  */
  void* first_cov;      /* T[max_tracks][36] SMOOTHED covariance at the first measurement                     */
  void* entry_params;   /* T[max_track_entries][6] SMOOTHED parameters at every measurement, parallel to
                           ckf_tracks.meas_idx (entry track_offsets[t] is the first measurement of track t)  */
  int64_t* work;        /* [4] or NULL: the call ADDS its RKN4 trials, accepted steps, module-to-module moves and
                           Kalman updates here (zero it before the call; roofline accounting)    */
  int32_t smoother_precision; /* INPUT.  0 or 64: the RTS recursion runs in float64 (the product's choice, K5).
                           32 (handles of precision 32 only): it runs in float32 -- kept to study the instability
                           of the float32 smoother that PAPER.md:61, :100 report, not for production             */
  int32_t n_tracks_upper; /* INPUT.  0, or a host-side upper bound on *tracks->n_tracks (e.g. from a previous read-back):
                           passes of the state store beyond it are not enqueued at all (without it every pass up to
                           max_tracks is enqueued and those beyond the device's count return at once)                */
  int32_t smoother;     /* INPUT.  0: RTS recursion (K4).  1: two-filter "optimal" smoother (K4'): the
                           forward-filtered state combined with a backward information filter over the same stored
                           states; same result (tested), no differences of nearly equal covariances                 */
} ckf_fits;

/* Fits every candidate of `tracks` (the DEVICE arrays a ckf_find on the same measurements and seeds filled;
 * *tracks->n_tracks is read on the device, no host synchronisation).  Asynchronous on `cuda_stream`; allocates
 * nothing: the state store was reserved by ckf_create (config.max_fit_tracks; CKF_E_CAPACITY if that was 0).  All
 * candidates are fitted, in passes of the store's size.  Calls on different streams are ordered one after the other
 * (one state store per handle). */
int ckf_fit(ckf_handle* handle, const ckf_measurements* measurements, const ckf_seeds* seeds, const ckf_tracks* tracks,
            ckf_fits* out, void* cuda_stream);

/* ---- Ambiguity resolution after the CKF ----------------------------------
 * "Duplicate tracks arise when multiple tracks share the same or very similar hit patterns ... an additional
 * algorithm -- known as ambiguity resolution -- will be integrated into the reconstruction chain to remove such tracks
 * after the CKF stage".  The paper gives no algorithm; rules AR1-AR3 of DESIGN.md 3 define a greedy
 * shared-hit resolver: candidates are ranked by (more measurements, smaller chi2_sum rounded to float32, lower
 * index); visited in that order, a candidate is ACCEPTED iff the number s of its measurements that already belong to
 * accepted candidates satisfies s <= max_shared_hits and s <= max_shared_fraction * n_meas; an accepted candidate
 * takes its free measurements.  The result equals that sequential greedy exactly and is deterministic.
 * DEVICE pointers, caller-owned, sized from max_tracks. */
typedef struct {
  int32_t* accepted;           /* [max_tracks] 1 = kept, 0 = removed                                        */
  int32_t* n_shared;           /* [max_tracks] s of the candidate's decision                                */
  int32_t* summary;            /* [2] number of accepted candidates, rounds the parallel resolution took    */
  int32_t max_shared_hits;     /* INPUT                                                                      */
  double max_shared_fraction;  /* INPUT; 1.0 = no fractional limit                                           */
} ckf_resolution;

/* Resolves the candidates of `tracks` (the DEVICE arrays ckf_find filled; *tracks->n_tracks is read on the device).
 * n_measurements = ckf_measurements.n of that find.  Asynchronous on `cuda_stream`, allocates nothing (20 bytes per
 * measurement and 12 per candidate were reserved by ckf_create); at most 2^24 candidates.  Calls on different streams
 * are ordered one after the other (one workspace per handle). */
int ckf_resolve(ckf_handle* handle, const ckf_tracks* tracks, int32_t n_measurements, ckf_resolution* out,
                void* cuda_stream);

/* ---- ckf_resolve for callers that may not allocate --------------------------------------------------------------------
 * The same resolution (same kernel, same rules AR1-AR3, same results) WITHOUT a handle and without any allocation: no
 * cudaMalloc / cudaFree / allocating library routine is called, at set-up or later, so it may be used under CUDA graph
 * capture, in serving loops and in harnesses that forbid allocation.  Its scratch (rank keys, per-measurement minima,
 * owners, states) lives in a static __device__ array of the library, CKF_RESOLVE_STATIC_SCRATCH_BYTES (3.25 MiB) on
 * every GPU that loads the library, held until the process exits.  Hence the limits: at most
 * CKF_RESOLVE_STATIC_MAX_TRACKS candidates and CKF_RESOLVE_STATIC_MAX_MEASUREMENTS measurements; larger sizes are
 * rejected with CKF_E_CAPACITY and a message (use ckf_resolve).
 *   tracks          DEVICE arrays as filled by ckf_find; n_tracks, track_offsets, meas_idx, chi2_sum are read
 *   max_tracks      capacity of the caller's arrays (out->accepted, out->n_shared, tracks->chi2_sum): candidates beyond
 *                   it are ignored, as in ckf_resolve; 1 .. CKF_RESOLVE_STATIC_MAX_TRACKS
 *   n_measurements  ckf_measurements.n of the find; 0 .. CKF_RESOLVE_STATIC_MAX_MEASUREMENTS
 *   precision       32 or 64: element type of tracks->chi2_sum
 *   out             as for ckf_resolve (DEVICE arrays, caller-owned; limits are inputs)
 * Asynchronous on `cuda_stream`, which must belong to the CURRENT device (the array's address is looked up once per
 * device, on first use with that device current).  Every call shares the one array: the kernel re-initialises what it
 * reads, so calls in stream order need no clearing by the caller, but two calls that OVERLAP on the GPU (different
 * streams, no ordering between them) race and give garbage -- order them.  Errors: CKF_E_ARG, CKF_E_CAPACITY, CKF_E_CUDA;
 * text from ckf_last_error(NULL). */
#define CKF_RESOLVE_STATIC_MAX_TRACKS 65536
#define CKF_RESOLVE_STATIC_MAX_MEASUREMENTS 131072
#define CKF_RESOLVE_STATIC_SCRATCH_BYTES (CKF_RESOLVE_STATIC_MAX_TRACKS * 12 + CKF_RESOLVE_STATIC_MAX_MEASUREMENTS * 20 + 256)
int ckf_resolve_static(const ckf_tracks* tracks, int32_t max_tracks, int32_t n_measurements, int32_t precision,
                       ckf_resolution* out, void* cuda_stream);

/* ---- Triplet seeding + track-parameter estimation, the stage in front of the CKF ---
 * "The spacepoints are used in the seeding algorithm where triplets, a set of three spacepoints which can approximately
 * form a helix, are found.  In the track parameter estimation algorithm, the position and momentum of tracks, called a
 * seed, are estimated at the first spacepoint using the helix model".  The paper gives no cut and no
 * formula; rules S0-S6 of DESIGN.md 3: spacepoints = global positions of the measurements of three barrel layers;
 * doublets (inner, outer) with |dphi| <= dphi_max, |cot theta| <= cot_max, |z0| <= z0_max; triplets with
 * |cot(b,m) - cot(m,t)| <= dcot_max whose circle through the three transverse points has pT >= pt_min (field at the
 * bottom point) and passes within d0_max of the z axis; every such triplet is a seed: bound parameters on the bottom
 * measurement's module (its loc0, loc1; tangent direction, arc-length cot theta, charge from the turning sense, q/p) and
 * a diagonal covariance cov_scale x (measurement variances, sigma_angle^2 twice, what the sagitta resolves in q/p plus
 * (rel_sigma_qop q/p)^2, and 1 for t unscaled). */
typedef struct {
  int32_t layer_b;       /* barrel layers, bottom < middle < top */
  int32_t layer_m;
  int32_t layer_t;
  double dphi_max;       /* doublet cuts: rad                    */
  double cot_max;
  double z0_max;         /* mm                                   */
  double dcot_max;       /* triplet cuts                         */
  double pt_min;         /* GeV                                  */
  double d0_max;         /* mm                                   */
  double sigma_angle;    /* covariance recipe, see above         */
  double rel_sigma_qop;
  double cov_scale;
} ckf_seeding;

/* Seeds in the layout of ckf_seeds.  DEVICE pointers, caller-owned, sized from `capacity`.  Order: by (bottom, middle,
 * top) measurement index; deterministic.  *n_seeds is written on the device: read it (after the stream) to fill
 * ckf_seeds.n for ckf_find. */
typedef struct {
  int32_t* n_seeds;    /* [1]                                                                    */
  int32_t* status;     /* [1] 1 = more seeds than capacity (the first `capacity` are kept), 2 = the doublet lists did
                          not fit config.max_seed_doublets (no seed is reported)                 */
  int32_t* module_id;  /* [capacity] module of the bottom measurement                             */
  void* params;        /* T[capacity][6]                                                          */
  void* cov;           /* T[capacity][36]                                                         */
  int32_t* triplets;   /* [capacity][3] measurement indices (bottom, middle, top)                 */
  int32_t capacity;    /* INPUT                                                                   */
} ckf_seed_out;

/* Seeds of one event's measurements (DEVICE arrays as for ckf_find, one event).  Asynchronous on `cuda_stream`,
 * allocates nothing (CKF_E_CAPACITY if config.max_seed_doublets was 0).  Calls on different streams are ordered one
 * after the other (one workspace per handle). */
int ckf_seed(ckf_handle* handle, const ckf_measurements* measurements, const ckf_seeding* seeding, ckf_seed_out* out,
             void* cuda_stream);

/* Copies the work counters of the most recent ckf_find issued on `cuda_stream` (synchronises that stream). */
int ckf_get_counters(ckf_handle* handle, void* cuda_stream, ckf_counters* out);

/* Per-kernel device times of one ckf_find, summed over the levels (CUDA events on the call's stream). */
typedef struct {
  float init_ms;          /* per-event reset                                                            */
  float sort_ms;          /* gate index (slice sort)                                                    */
  float step_ms;          /* ckf_step: navigation + adaptive RKN4 + Jacobian transport (the hot kernel) */
  float visit_ms;         /* ckf_visit: arrival Jacobian, covariance transport, chi2 gate, k best       */
  float scan_ms;          /* ckf_scan: per-seed cap, emission records, child offsets                    */
  float update_ms;        /* ckf_update: Kalman update, link append, departure state                    */
  float emit_ms;          /* emission: seed scan, backtrace, finalize                                   */
  int32_t launches;       /* kernel launches of one ckf_find                                            */
} ckf_timing;

/* Measurement aid.  ckf_set_timing(handle, 1) makes every later ckf_find record a CUDA event after each
 * kernel and SYNCHRONISE its stream at the end (so it is off by default); ckf_get_timing returns the times of
 * the most recent timed ckf_find issued on `cuda_stream`. */
int ckf_set_timing(ckf_handle* handle, int on);
int ckf_get_timing(ckf_handle* handle, void* cuda_stream, ckf_timing* out);

/* Launch configuration chosen at ckf_create for the hot kernel (ckf_step: navigation + RKN4): thread blocks,
 * threads per block, shared bytes, registers per thread (any pointer may be NULL). */
int ckf_get_launch_info(const ckf_handle* handle, int32_t* blocks, int32_t* threads, int32_t* smem_bytes,
                        int32_t* regs);

/* Measurement aid: the plain-ALU FMA peak of the current device, the roofline denominator of this path (north_star:
 * "% of FP pipe peak"; the method does not use the tensor cores).  FMA chains in registers on every SM, launched back
 * to back for at least `seconds` on the default stream, synchronous.  mix 0: float32 chains only; 1: float64 only;
 * 2: 8 float32 + 4 float64 chains per thread at once.  *tflops_f32 / *tflops_f64: flop rates over the whole run (an
 * FMA counts 2); *best_f32 / *best_f64 (may be NULL): rates of the fastest single launch.  Needs no handle. */
int ckf_measure_alu_peak(int mix, double seconds, double* tflops_f32, double* tflops_f64, double* best_f32,
                         double* best_f64);

int ckf_destroy(ckf_handle* handle);

/* Text of the calling thread's last failed call (handle may be NULL; it is not used). */
const char* ckf_last_error(const ckf_handle* handle);

int ckf_abi_version(void);

#ifdef __cplusplus
}
#endif
#endif /* CKF_H_ */

/* =============================================================================================
 * tpc_b200.h -- C ABI of the B200-native TPC track-reconstruction hot path.
 *
 * What it is.  The data-parallel hot path of ALICE's Run-3 synchronous GPU processing: TPC track
 * reconstruction on a continuous-readout Time Frame (TF = 128 orbits, no event
 * boundaries; l.37, l.47: TPC tracking dominates the synchronous workload and has no a-priori
 * absolute z; l.102: cost grows with tracks x attached clusters).  The paper names the step but
 * never spells the algorithm out, so the operations are the four steps of BASELINE.json
 * `north_star` made concrete by the readings R1-R23 of SURVEY.md §8(c) (restated in DESIGN.md):
 *
 *   tpc_grid_build   step 1  (R7)        per-(sector,row) (y, zeta) search grid: stable counting
 *                                        sort by bin, bin start offsets
 *   tpc_find_tracks  steps 2,3a,4        cellular-automaton neighbours (R9), reciprocal links and
 *                    (R9-R20)            start hits (R10), Kalman following (R11-R18), one-shot
 *                                        selection with exclusive cluster assignment (R20)
 *   tpc_fit_tracks   step 3b (R21-R22)   3-point seed + outward/inward Kalman refit, fp32
 *   tpc_track_time   next     (R24)       per-track closest approach to the beam line, z0, time offset
 *   tpc_find_collisions next  (R25)       collisions = peaks of the per-track time offsets; track -> collision
 *
 * Conventions.
 *  - Every pointer is a DEVICE pointer unless its name ends in `_host`.  Every call only enqueues
 *    work on `stream` (a cudaStream_t passed as void*; NULL = the legacy default stream) and
 *    returns without synchronising.  The library never allocates or frees device memory: the
 *    caller owns every buffer, including the workspace.
 *  - Return value: TPC_OK (0) or a negative tpc_status_t.  Host-detectable misuse (NULL pointer,
 *    workspace too small, sizes out of range) is a return code and nothing is enqueued.  Problems
 *    found on the device (tracklet / track capacity overflow, cluster outside the grid's z range)
 *    set bits in counters[TPC_CNT_STATUS]; outputs are truncated, never written out of bounds.
 *  - Layout: external cluster data is SoA fp32 (one array per field) + int32 sector_row =
 *    sector*n_rows + row, in arbitrary order.  The workspace holds the library's internal state
 *    (sorted 16-byte cluster records, bin offsets, links, tracklet tables) and is laid out as a
 *    pure function of (params, n_clusters, max_tracklets): the same three values must be passed
 *    to tpc_workspace_bytes, tpc_grid_build and tpc_find_tracks.  The grid inside it is valid
 *    until the next tpc_grid_build on the same workspace.
 *  - All cluster indices in outputs are ORIGINAL indices (positions in the caller's arrays).
 *  - Arithmetic: IEEE fp32, one rounding per written operation (compiled without FMA
 *    contraction) so that results are reproducible bit for bit; integer work is exact and every
 *    arg-min/arg-max breaks ties by original cluster index, so the output is deterministic.
 * ============================================================================================= */
#ifndef TPC_B200_H_
#define TPC_B200_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define TPC_MAX_ROWS 152
#define TPC_MAX_TRACKLETS 33554432 /* 2^25 */

typedef enum {
  TPC_OK = 0,
  TPC_EINVAL = -1,     /* NULL pointer, negative size, n_rows/n_sectors out of range, bins >= 2^31 */
  TPC_ENOMEM_WS = -2,  /* ws_bytes smaller than tpc_workspace_bytes() for these sizes */
  TPC_ECUDA = -3,      /* a CUDA runtime call failed at enqueue time (see tpc_last_cuda_error) */
  TPC_ELIMIT = -4      /* a size beyond the fixed scratch array of a *_static entry point (tpc_pair_sides_static) */
} tpc_status_t;

/* indices into the int32 counters[TPC_N_COUNTERS] device array written by tpc_find_tracks */
enum {
  TPC_CNT_TRACKS = 0,     /* K  = number of accepted tracks (clamped to max_tracks)            */
  TPC_CNT_TRACKLETS = 1,  /* S  = number of start hits followed (clamped to max_tracklets)      */
  TPC_CNT_HITS = 2,       /* sum of trk_nhits over the K tracks = entries used in trk_hits      */
  TPC_CNT_STATUS = 3,     /* bit mask of TPC_ST_*                                               */
  TPC_CNT_STARTS_FOUND = 4, /* start hits found before clamping                                 */
  TPC_CNT_TRACKS_FOUND = 5, /* accepted tracks before clamping                                  */
  TPC_CNT_FOLLOWED_DOWN = 6, /* tracklets that went on to the downward leg (start hit not picked up by an upward leg, R17) */
  TPC_CNT_RESERVED7 = 7,
  TPC_CNT_PROP_LO = 8,    /* follower work (time ~ tracks x attached clusters):      */
  TPC_CNT_PROP_HI = 9,    /*   64-bit count of helix transports (R12) done by the follower, lo/hi    */
  TPC_CNT_UPD_LO = 10,    /*   64-bit count of Kalman updates (R13) done by the follower, lo/hi      */
  TPC_CNT_UPD_HI = 11,
  TPC_CNT_CAND_LO = 12,   /*   64-bit count of candidate clusters chi2-tested in R16 searches, lo/hi */
  TPC_CNT_CAND_HI = 13,
  TPC_CNT_CLAIMS_LO = 14, /*   64-bit count of hits recorded by the tracklets of TPC_CNT_FOLLOWED_DOWN (R18), lo/hi */
  TPC_CNT_CLAIMS_HI = 15,
  TPC_N_COUNTERS = 16
};
#define TPC_ST_TRACKLET_OVERFLOW 1 /* more start hits than max_tracklets: the excess was dropped */
#define TPC_ST_TRACK_OVERFLOW 2    /* more accepted tracks than max_tracks: the excess was dropped */
#define TPC_ST_Z_CLAMPED 4         /* a cluster lay outside [z_lo,z_hi] and was put in an edge bin */
#define TPC_ST_BAD_ROW 8           /* a sector_row outside [0, n_sectors*n_rows): that cluster is in no grid bin, no
                                      search sees it, it stays unassigned (cluster_track = -1)            */

/* Host POD, passed by pointer and copied during the call.  Every field is an input of the method
 * (SURVEY.md §8(b),(c)): geometry R1-R2, field constant R4, measurement errors R6, grid cell R7,
 * cuts R9-R22.  Defaults in parentheses. */
typedef struct {
  int32_t n_sectors;             /* 36 (18 per side; sectors >= 18 have side = -1), or 1         */
  int32_t n_rows;                /* <= TPC_MAX_ROWS (152)                                         */
  float row_x[TPC_MAX_ROWS];     /* sector-local x of pad row r, cm, strictly increasing (R1)     */
  float tan_half;                /* tan(10 deg): row r spans |y| <= row_x[r]*tan_half (R1)        */
  float kB;                      /* 0.299792458e-2 * B[T]; dphi/ds = -kB*q/pT (R4)                */
  float sigma_y, sigma_z;        /* cluster errors, cm (0.08, 0.10) (R6)                          */
  float z_lo, z_hi;              /* range of zeta = side*z covered by the grid, cm (R7)           */
  float cell_y, cell_z;          /* grid cell, cm (R7)                                            */
  float ca_max_dydx, ca_max_dzdx, ca_cut;                 /* R9  (2.0, 2.5, 20)                   */
  float chi2_cut, chi2_chain_cut, win_max;                /* R15-R16 (16, 30, 5 cm)               */
  float max_sinphi, edge_margin;                          /* R12, R16 (0.95, 1 cm)                */
  int32_t max_gap, min_hits, n_fit_passes;                /* R16, R20, R22 (4, 10, 2); min_hits >= 3 (R21) */
  float cov0[5];                 /* initial covariance diagonal (1,1,1,10,100) (R14, R22)         */
} tpc_params_t;

/* Human-readable text for a tpc_status_t (static storage). */
const char* tpc_strerror(int status);
/* Text of the last CUDA runtime error seen by this thread's last failing call (static storage). */
const char* tpc_last_cuda_error(void);
/* Library version, e.g. "0.1.0". */
const char* tpc_version(void);

/* Number of grid bins for these parameters: n_sectors * sum_r ny_r * nz (R7).  Host only.
 * Returns TPC_EINVAL if params are inconsistent or the count does not fit in int32. */
int tpc_grid_bins(const tpc_params_t* params_host, int64_t* n_bins_host);

/* Bytes of workspace needed for n_clusters clusters and at most max_tracklets start hits.
 * max_tracklets <= TPC_MAX_TRACKLETS (the tracklet number shares the 64-bit R20 selection key
 * with nHits and the start index); larger values are TPC_EINVAL in every workspace-taking call. */
int tpc_workspace_bytes(const tpc_params_t* params_host, int64_t n_clusters, int64_t max_tracklets,
                        size_t* bytes_host);

/* Step 1 (R7).  Sorts the n clusters into the grid held in `workspace`.
 *   y, z, sector_row : [n] inputs, arbitrary order; must stay alive and unmodified until the last
 *                      call that uses this grid has completed on `stream`.
 *   x, q             : [n] pad-row x and cluster charge; carried by the interface (BASELINE.json
 *                      "fp32 (x,y,z,row,charge) clusters") but not read: x == row_x[row] by
 *                      construction and the tracker does not use charge.  May be NULL.
 * n == 0 is legal.  Clusters outside [z_lo,z_hi] are clamped into the edge bins (status bit is
 * raised later by tpc_find_tracks' counters; results stay exact because searches re-check cm). */
int tpc_grid_build(const tpc_params_t* params_host, int64_t n_clusters, int64_t max_tracklets,
                   const float* x, const float* y, const float* z, const float* q,
                   const int32_t* sector_row, void* workspace, size_t ws_bytes, void* stream);

/* Debug/parity view of the grid (R7): original indices in sorted order and bin offsets.
 * sorted_idx [n] and/or bin_first [n_bins+1] may be NULL.  Enqueues device-to-device copies. */
int tpc_grid_export(const tpc_params_t* params_host, int64_t n_clusters, int64_t max_tracklets,
                    const void* workspace, size_t ws_bytes, int32_t* sorted_idx, int32_t* bin_first,
                    void* stream);

/* Steps 2, 3a, 4 (R9-R20) on the grid built by tpc_grid_build in the same workspace.
 *   cluster_track [n]           : track index (0..K-1) owning each cluster, -1 = none (R20)
 *   trk_seed      [max_tracks]  : original index of the track's start hit (unique per track)
 *   trk_sector    [max_tracks]  : sector of the track
 *   trk_nhits     [max_tracks]  : hits kept after arbitration (>= min_hits)
 *   trk_first_hit [max_tracks]  : offset of the track's first hit in trk_hits
 *   trk_hits      [n]           : original cluster indices, row-ascending per track
 *   counters      [TPC_N_COUNTERS] int32, see TPC_CNT_*
 * Track order is deterministic (ascending grid position of the start hit) but carries no meaning:
 * match tracks by trk_seed. */
int tpc_find_tracks(const tpc_params_t* params_host, int64_t n_clusters, int64_t max_tracklets,
                    void* workspace, size_t ws_bytes, int32_t* cluster_track, int64_t max_tracks,
                    int32_t* trk_seed, int32_t* trk_sector, int32_t* trk_nhits,
                    int64_t* trk_first_hit, int32_t* trk_hits, int32_t* counters, void* stream);

/* Debug/parity view of the intermediate stages of the last tpc_find_tracks on this workspace,
 * all in ORIGINAL cluster indices (-1 = none).  Any output pointer may be NULL.
 *   link_up, link_dn [n]  : R9 raw links;  up_c, dn_c [n] : R10 cleaned links
 *   starts [max_tracklets]: start hit of tracklet t;  tl_nhits [max_tracklets]: hits recorded
 *   row_hit [TPC_CNT_TRACKLETS * n_rows] : row_hit[t*n_rows + r] (R18), row-major per tracklet
 * Entries for t >= counters[TPC_CNT_TRACKLETS] are left untouched. */
int tpc_find_export(const tpc_params_t* params_host, int64_t n_clusters, int64_t max_tracklets,
                    const void* workspace, size_t ws_bytes, int32_t* link_up, int32_t* link_dn,
                    int32_t* up_c, int32_t* dn_c, int32_t* starts, int32_t* tl_nhits,
                    int32_t* row_hit, void* stream);

/* Step 3b (R21-R22).  Refit of K = counters[TPC_CNT_TRACKS] hit lists (read on the device; the
 * call never synchronises).
 *   workspace != NULL : must be the workspace on which tpc_find_tracks produced exactly these
 *                       trk_nhits / trk_first_hit / trk_hits (same n_clusters, max_tracklets).
 *                       tpc_find_tracks stored the (y, z, row) of every hit in hit-list order
 *                       there; the fit streams those records instead of gathering, and y, z,
 *                       sector_row, trk_hits are not read (may be NULL).  K is clamped to the
 *                       tracklet capacity of that workspace (find cannot have produced more).
 *   workspace == NULL : self-contained gather through y, z, sector_row (the caller's arrays,
 *                       original order) and trk_hits, so any hit lists can be refitted, e.g.
 *                       truth hits; max_tracklets and ws_bytes are ignored.
 * Both paths run the same arithmetic and give bit-identical results.
 *   par [5][max_tracks]  : y, dz = z - zref, sinphi, tanlambda, q/pT at x = xref   (SoA)
 *   cov [15][max_tracks] : lower triangle, row-major (00,10,11,20,21,22,...)       (SoA)
 *   xref, zref, chi2 [max_tracks], ndf [max_tracks] (= 2*nhits-5; chi2 = -1, ndf = -1 if the
 *   propagation left |sinphi| <= max_sinphi). */
int tpc_fit_tracks(const tpc_params_t* params_host, int64_t n_clusters, int64_t max_tracklets,
                   void* workspace, size_t ws_bytes, const float* y, const float* z,
                   const int32_t* sector_row, const int32_t* counters, int64_t max_tracks,
                   const int32_t* trk_nhits, const int64_t* trk_first_hit, const int32_t* trk_hits,
                   float* par, float* cov, float* xref, float* zref, float* chi2, int32_t* ndf,
                   void* stream);

/* After the hot path (R24; tracks are assigned to collisions only
 * after the reconstruction).  For each of the K = counters[TPC_CNT_TRACKS] fitted tracks: the point of closest
 * approach of its helix to the beam line (origin of the sector-local frames), in fp64 from the fp32 state:
 *   phi0 [max_tracks] : global azimuth of the direction of flight there, [0, 2 pi)
 *   z0   [max_tracks] : z there (same frame as the input z: includes the drift-time shift), cm
 *   dca  [max_tracks] : distance of closest approach in the bending plane, cm (>= 0)
 *   t0   [max_tracks] : time offset -side*z0/v_drift in microseconds for v_drift in cm/us (R5): the collision
 *                       time of a primary from a vertex at z = 0
 * par, xref, zref, trk_sector are the outputs of tpc_fit_tracks / tpc_find_tracks.  Enqueue only. */
int tpc_track_time(const tpc_params_t* params_host, const int32_t* counters, int64_t max_tracks,
                   const int32_t* trk_sector, const float* par, const float* xref, const float* zref,
                   float v_drift, float* phi0, float* z0, float* dca, float* t0, void* stream);

/* Collisions from the per-track time offsets (R25).  Integer work on
 * a time histogram of n_bins bins of bin_width [us] starting at t_lo:
 *   used tracks: finite t0, dca <= dca_max, t_lo <= t0 < t_lo + n_bins*bin_width, on the selected TPC side
 *                (side_sel = +1: sectors < 18, -1: sectors >= 18, 0: both; trk_sector may be NULL for 0).  The two sides
 *                see a collision at t -/+ z_vertex/v_drift (R5), so they are clustered separately and paired afterwards;
 *   s[b] = tracks in bins b-2..b+2;  bin b is a collision iff s[b] >= n_min, s[b] > s[b-j] and s[b] >= s[b+j], j = 1..3;
 *   coll_time [max_collisions]    : mean t0 of the tracks in the collision's 5 bins (exact: accumulated as
 *                                   round(1024 (t0 - t_lo)) in int64), collisions in ascending time order
 *   coll_ntracks, coll_bin [max_collisions] : tracks in those 5 bins; the peak bin
 *   trk_collision [max_tracks]    : nearest collision within 5 bins of the track's bin (ties: the earlier), -1 = none
 *   n_collisions [2] (device)     : collisions found; collisions written (clamped to max_collisions)
 * K = counters[TPC_CNT_TRACKS] is read on the device.  workspace: tpc_collisions_workspace_bytes(n_bins,
 * max_tracks) bytes, 256-byte aligned, caller-owned.  Enqueue only. */
int tpc_collisions_workspace_bytes(int64_t n_bins, int64_t max_tracks, size_t* bytes_host);
int tpc_find_collisions(const int32_t* counters, int64_t max_tracks, const float* t0, const float* dca,
                        const int32_t* trk_sector, int32_t side_sel, double t_lo, double bin_width, int64_t n_bins, double dca_max, int32_t n_min,
                        void* workspace, size_t ws_bytes, int64_t max_collisions, float* coll_time,
                        int32_t* coll_ntracks, int32_t* coll_bin, int32_t* trk_collision,
                        int32_t* n_collisions, void* stream);

/* Pairing of the two sides' collisions into (t, z_vertex) (last part; R29).  Inputs: the
 * outputs of two tpc_find_collisions calls, side_sel = +1 (`_a`) and -1 (`_c`): n_collisions [2], coll_time,
 * coll_ntracks (device; the number written, n_collisions[1], is read on the device).  A collision at time t with
 * vertex z_v is seen at t - z_v/v_drift by side A and at t + z_v/v_drift by side C.  (i, j) is admissible iff
 * |t_c[j] - t_a[i]| <= dt_max; cost = ((t_c - t_a) / sigma_t)^2 + (n_a - n_c)^2 / (n_a + n_c + 1) in double; pairs are
 * the reciprocal arg-mins (ties: the lower index).  Outputs (device): pair_of_a, pair_of_c [max_collisions] (partner
 * or -1), t, z_vertex [max_collisions] per pair in ascending side-A index (t = (t_a + t_c)/2, z_vertex =
 * v_drift (t_c - t_a)/2), n_pairs [1].  workspace: tpc_pair_sides_workspace_bytes(max_collisions), 256-byte aligned.
 * max_collisions is the capacity of every per-collision array passed here; a side whose list holds more
 * (n_collisions[1] > max_collisions, e.g. tpc_find_collisions was given a larger capacity) is read up to its first
 * max_collisions entries only -- the lists are in time order, so the later collisions stay unpaired -- and nothing is
 * written beyond that capacity.  max_collisions <= 2147483000.  Enqueue only. */
int tpc_pair_sides_workspace_bytes(int64_t max_collisions, size_t* bytes_host);
int tpc_pair_sides(const int32_t* n_collisions_a, const float* coll_time_a, const int32_t* coll_ntracks_a,
                   const int32_t* n_collisions_c, const float* coll_time_c, const int32_t* coll_ntracks_c,
                   int64_t max_collisions, double dt_max, double sigma_t, double v_drift, void* workspace,
                   size_t ws_bytes, int32_t* pair_of_a, int32_t* pair_of_c, float* t, float* z_vertex,
                   int32_t* n_pairs, void* stream);

/* tpc_pair_sides without a workspace, for callers that cannot allocate device memory.
 * Who that is: code that runs where cudaMalloc is not allowed or not wanted -- a processing step inside a framework
 * that hands out all GPU memory itself from one big pre-allocated block (the online processing keeps
 * reusing one block of GPU memory for its consecutive processing steps, sized so that a whole Time Frame fits), a callback or a thread
 * that must not take the allocator's device-wide lock or cause the implicit synchronisation a cudaMalloc / cudaFree
 * brings, a process whose memory budget was handed out completely at start-up.  Such a caller has device buffers for
 * its inputs and outputs but no spare block to pass as `workspace` and no way to get one.
 * What it does: exactly tpc_pair_sides (same kernels, same arithmetic, same outputs bit for bit), with the two
 * arg-min tables best_c / best_a -- the only scratch memory that operation needs -- placed in an array that is part of
 * the library image: 2 x 65 792 bytes = 128.5 KiB of device memory on every GPU that loads the library, held until
 * the process exits.  The caller passes inputs and outputs only; the call makes no cudaMalloc, cudaFree or any
 * other allocating call (it does not create events either: its three launches are counted by tpc_profile_collect
 * but never timed).
 * Limit: max_collisions <= TPC_PAIR_SIDES_STATIC_MAX (16 384 collisions per side; a 128-orbit Time Frame at 50 kHz
 * holds about 570).  A larger value returns TPC_ELIMIT and enqueues nothing; use tpc_pair_sides with a workspace of
 * your own for that.  As for tpc_pair_sides, a list longer than max_collisions is read up to its first
 * max_collisions entries, so the array is never overrun whatever the device-side counts say.
 * First call on a device: the library looks up the device address of the array once per device (with the
 * caller's current device; cudaGetSymbolAddress, which may also make the CUDA runtime load the library's
 * kernels on that device).  Make this first call during set-up, outside any stream capture; an easy way is one call
 * with empty lists (n_collisions_*[1] = 0).  Later calls on that device only launch the three kernels on `stream`.
 * Sharing: all calls on one GPU use the same array -- from every stream, every host thread and every library user in
 * the process.  Nothing in it has to start at zero (each call overwrites the entries it later reads), so there is
 * nothing to clear between calls; but two calls whose kernels can overlap on the GPU (different streams without an
 * event between them) race on it and give wrong pairs.  Keep all calls on one stream, or order them with events.
 * Errors: TPC_EINVAL as tpc_pair_sides; TPC_ELIMIT as above; TPC_ECUDA if the address look-up or a launch fails. */
#define TPC_PAIR_SIDES_STATIC_MAX 16384
int tpc_pair_sides_static(const int32_t* n_collisions_a, const float* coll_time_a, const int32_t* coll_ntracks_a,
                          const int32_t* n_collisions_c, const float* coll_time_c, const int32_t* coll_ntracks_c,
                          int64_t max_collisions, double dt_max, double sigma_t, double v_drift, int32_t* pair_of_a,
                          int32_t* pair_of_c, float* t, float* z_vertex, int32_t* n_pairs, void* stream);

/* ---- host-buffer entry points (bench.py `e2e`; a continuous stream of Time Frames through
 * reused GPU memory) ---------------------------------------------------------------------------------------------
 * tpc_result_t names the outputs of tpc_find_tracks + tpc_fit_tracks (layouts as documented there).  The same
 * struct describes the DEVICE buffers of a tracking context and the pinned HOST buffers the results are copied to;
 * in the host struct a NULL member is not copied (counters is required). */
typedef struct {
  int32_t* cluster_track;   /* [n_clusters] */
  int32_t* trk_seed;        /* [max_tracks] */
  int32_t* trk_sector;      /* [max_tracks] */
  int32_t* trk_nhits;       /* [max_tracks] */
  int64_t* trk_first_hit;   /* [max_tracks] */
  int32_t* trk_hits;        /* [n_clusters] */
  int32_t* counters;        /* [TPC_N_COUNTERS] */
  float* par;               /* [5][max_tracks] */
  float* cov;               /* [15][max_tracks] */
  float* xref;              /* [max_tracks] */
  float* zref;              /* [max_tracks] */
  float* chi2;              /* [max_tracks] */
  int32_t* ndf;             /* [max_tracks] */
} tpc_result_t;

/* tpc_track_host_async: enqueue only.  Copies y, z, sector_row host->device into the caller's staging buffers,
 * runs tpc_grid_build, tpc_find_tracks, tpc_fit_tracks into `dev`, and copies back what has a size known to the
 * host: counters and (if host->cluster_track) cluster_track [n_clusters].  Returns without synchronising, so that a
 * caller with two contexts on two streams overlaps the host->device copy of one Time Frame with the tracking of
 * the previous one and the device->host copies of the one before.  Host buffers must be pinned and stay
 * untouched until `stream` has passed this call's work.
 * tpc_track_host_fetch: to be called once host->counters has arrived (cudaEventSynchronize on an event recorded
 * after tpc_track_host_async, or a stream synchronise).  Reads K = counters[TPC_CNT_TRACKS] and H =
 * counters[TPC_CNT_HITS] from host->counters and enqueues device->host copies of exactly the first K entries of
 * every per-track array (rows of par / cov keep their pitch of max_tracks) and the first H entries of trk_hits, for
 * every non-NULL member of `host`.  bytes_host (may be NULL) receives the bytes it enqueued.
 * tpc_track_host: tpc_track_host_async, synchronise, tpc_track_host_fetch, synchronise.
 * All three: TPC_EINVAL for missing buffers; otherwise the return codes of the three steps. */
int tpc_track_host_async(const tpc_params_t* params_host, int64_t n_clusters, int64_t max_tracklets,
                         int64_t max_tracks, const float* y_host, const float* z_host,
                         const int32_t* sector_row_host, float* y_dev, float* z_dev, int32_t* sector_row_dev,
                         void* workspace, size_t ws_bytes, const tpc_result_t* dev, const tpc_result_t* host,
                         void* stream);
int tpc_track_host_fetch(int64_t max_tracks, const tpc_result_t* dev, const tpc_result_t* host,
                         int64_t* bytes_host, void* stream);
int tpc_track_host(const tpc_params_t* params_host, int64_t n_clusters, int64_t max_tracklets,
                   int64_t max_tracks, const float* y_host, const float* z_host,
                   const int32_t* sector_row_host, float* y_dev, float* z_dev, int32_t* sector_row_dev,
                   void* workspace, size_t ws_bytes, const tpc_result_t* dev, const tpc_result_t* host,
                   void* stream);

/* ---- physics options of the refit and cluster tags ("removal of hits of tracks
 * not used for physics"; R28) -------------------------------------------------------------------------
 * tpc_fit_tracks_physics: tpc_fit_tracks (same workspace rule: workspace != NULL streams the track-ordered hit records
 * tpc_find_tracks left there and reads neither y, z nor trk_hits; workspace == NULL gathers through y, z, sector_row,
 * trk_hits and ignores max_tracklets / ws_bytes; both bit-identical; sector_row is needed either way, for the TPC
 * side) with the options of tpc_fit_options_t (host struct, read during the call):
 *   R28a x0inv > 0: multiple-scattering process noise after every transport over a path of L cm,
 *        theta0^2 = (0.0136 GeV)^2 (q/pT)^2 / (1 + tanl^2) L x0inv (x0inv = 1 / radiation length, per cm), added to the
 *        covariance of sinphi, tanlambda and q/pT;
 *   R28b outlier_cut > 0: in the last pass a hit whose chi2 against the predicted state exceeds it is left out:
 *        hit_flag = 1, ndf loses 2;
 *   R28d dedx > 0 (GeV per cm of path, beta = 1): after every transport q/pT changes by dq = (dedx |arc| |q/pT|) q/pT,
 *        added in the outward passes (a track is taken to fly outward and lose momentum), subtracted in the inward
 *        ones; C44 += (eloss_sigma dq)^2;
 *   R28e cluster errors at the predicted state (s = sinphi, tl = tanlambda) and the hit's drift length d:
 *        sigma_y^2 = sigma_y^2 (1 + err_ang_y s^2 / (1 - s^2)) + err_drift_y d,
 *        sigma_z^2 = sigma_z^2 (1 + err_ang_z tl^2) + err_drift_z d,   d = max(0, z_len - |z + side v_drift t0|),
 *        side = +1 for sectors < 18 else -1, t0 = trk_t0[track] (device, [max_tracks], the time offsets
 *        tpc_track_time writes; NULL or a NaN entry: no drift terms).
 * hit_flag [n_clusters], in hit-list order (same indexing as trk_hits), is always written (0 = used).  All options 0
 * (outlier_cut <= 0) give tpc_fit_tracks' results bit for bit.  TPC_EINVAL for a NULL options pointer, a negative,
 * infinite or NaN option (outlier_cut: NaN only), or missing buffers.
 * tpc_tag_clusters: tag [n_clusters] (uint8): bit 0 = attached to a track; bit 1 = that track is not used for
 * physics: ndf < 0 or |q/pT| = |par[4][track]| > qpt_max (low-pT loopers); bit 2 = rejected by R28b (hit_flag may be
 * NULL: bit 2 is then never set); 0 = unattached.  H = counters[TPC_CNT_HITS] is read on the device.  Enqueue only. */
typedef struct {
  float x0inv, outlier_cut;                              /* R28a, R28b */
  float dedx, eloss_sigma;                               /* R28d */
  float err_ang_y, err_ang_z, err_drift_y, err_drift_z;  /* R28e */
  float v_drift, z_len;                                  /* cm/us, cm: drift length of R28e */
} tpc_fit_options_t;
int tpc_fit_tracks_physics(const tpc_params_t* params_host, int64_t n_clusters, int64_t max_tracklets,
                           void* workspace, size_t ws_bytes, const float* y, const float* z,
                           const int32_t* sector_row, const int32_t* counters, int64_t max_tracks,
                           const int32_t* trk_nhits, const int64_t* trk_first_hit, const int32_t* trk_hits,
                           const tpc_fit_options_t* options_host, const float* trk_t0, float* par, float* cov,
                           float* xref, float* zref, float* chi2, int32_t* ndf, uint8_t* hit_flag, void* stream);
int tpc_tag_clusters(int64_t n_clusters, const int32_t* cluster_track, const int32_t* counters, int64_t max_tracks,
                     const float* par, const int32_t* ndf, const int32_t* trk_hits, const uint8_t* hit_flag,
                     double qpt_max, uint8_t* tag, void* stream);

/* ---- clusterizer (the step that feeds the tracker; R27) --------
 * Clusters from zero-suppressed digits (sector_row, pad, time_bin, adc), any order; two digits of one cell add up;
 * a digit with sector_row outside [0, n_sectors*n_rows), pad outside [0, 65535] or time_bin outside [0, 2^24) is
 * ignored, and so is one with adc <= 0 (not a zero-suppressed digit; every cell sum and S stay positive).  A cell of ADC >= peak_min is a peak iff it is strictly above its four earlier neighbours (time_bin - 1 at
 * pad - 1, pad, pad + 1; pad - 1 at the same time) and at least equal to the four later ones (missing = 0).  A peak
 * gives one cluster from the integer sums over its 3 x 3 cells, S = sum a, Sp = sum a dpad, St = sum a dtime:
 *   y = ((pad + 0.5) + Sp/S) pad_width - ymax_row,  zeta = ((time_bin + 0.5) + St/S) time_width + z_lo,
 *   z = zeta on side A (sectors < 18), -zeta on side C;  q = S           (fp32, one rounding per operation)
 * Outputs (device, [max_clusters]): y, z, q and sector_row -- what tpc_grid_build takes -- plus the peak cell out_pad /
 * out_time.  The SET of clusters is deterministic; their ORDER is the order in which the peaks were found and changes
 * from run to run.  tpc_find_tracks breaks exact ties by input index, so a caller that needs tracks reproducible to the
 * last tie orders the clusters by (sector_row, out_time, out_pad) -- unique per cluster -- before tpc_grid_build; n_clusters [2] (device): clusters found; clusters written
 * (= min(found, max_clusters)).  workspace: tpc_clusterize_workspace_bytes(n_digits) bytes, 256-byte aligned,
 * caller-owned.  Enqueue only.  TPC_EINVAL for missing buffers, n_digits > 2^31, pad_width / time_width <= 0,
 * peak_min < 1; TPC_ENOMEM_WS for a short workspace. */
int tpc_clusterize_workspace_bytes(int64_t n_digits, size_t* bytes_host);
int tpc_clusterize(const tpc_params_t* params_host, int64_t n_digits, const int32_t* sector_row, const int32_t* pad,
                   const int32_t* time_bin, const int32_t* adc, float pad_width, float time_width, int32_t peak_min,
                   void* workspace, size_t ws_bytes, int64_t max_clusters, float* y, float* z, float* q,
                   int32_t* out_sector_row, int32_t* out_pad, int32_t* out_time, int32_t* n_clusters, void* stream);

/* ---- merging of the sector-local tracks ("full tracking in the TPC", l.60;
 * DESIGN.md R26) ------------------------------------------------------------------------------------------------
 * tpc_find_tracks leaves a particle that crosses a 20-degree sector edge, the central electrode or a hole longer than
 * max_gap as several tracks.  tpc_merge_tracks links them and refits the merged hit lists:
 *   B can follow A iff B's sector is A's, an azimuthal neighbour on the same side or the mirror sector across the
 *   electrode; 1 <= first row of B - last row of A <= max_rows; |z_B - z_A| <= dz_max between the two ends
 *   (|z_B + z_A| across the electrode: the sides measure z_true -+ v_d t); tanlambda and q/pT differ by no more than
 *   d^2 <= 4 chi2_cut (C_A + C_B) each (a necessary condition of the cut); and chi2 < chi2_cut, chi2 = d^T S^-1 d over
 *   (y, z, sinphi, tanlambda, q/pT) between A's state -- transported by R12 to its outermost hit, rotated into B's
 *   frame, transported to B's innermost hit -- and B's state, S the sum of the two covariances.  Across the electrode
 *   z is left out (free time offset) and |z_A' + z_B| <= ce_tol + 2 |tanlambda_B| dx / cosphi_B is required instead.
 *   Links are the reciprocal arg-mins (ties: lowest trk_seed); global tracks are the chains of links.
 * Inputs: `dev` = the outputs of tpc_find_tracks + tpc_fit_tracks (cluster_track, trk_hits, counters of the struct are
 * not read; counters is passed separately), find_workspace = the workspace of that tpc_find_tracks call (its cached
 * hit records are read).  merge_workspace: tpc_merge_workspace_bytes(params, max_tracks) bytes, 256-byte aligned.
 * Outputs (device, caller-owned, `out`):
 *   trk_succ, trk_pred [max_tracks] : linked successor / predecessor of a track, -1 = none
 *   trk_succ_chi2 [max_tracks]      : chi2 of the best candidate successor (before reciprocity), -1 = none
 *   trk_global [max_tracks]         : global track of a sector-local track
 *   n_global [4]                    : global tracks M; links; pairs that passed the windows and the gate; pairs not
 *                                     tested because the pair list (4 max_tracks entries) was full.  n_global[3] is the
 *                                     overflow word of this call, as TPC_CNT_STATUS is for tpc_find_tracks: it is 0 on
 *                                     every workload seen so far (0.4 pairs per track on the bench Time Frame); when it is
 *                                     not, which pairs were left out depends on arrival order, so the links are
 *                                     incomplete and not reproducible -- treat it as an error and retry with a larger
 *                                     max_tracks (the Python binding raises)
 *   g_head, g_nseg, g_nhits [max_tracks] : first (innermost) piece, pieces and hits of global track g < M, in
 *                                     ascending order of g_head
 *   gpar [5][max_tracks], gcov [15][max_tracks], gxref, gzref, gchi2, gndf [max_tracks] : refit of the merged hit
 *                                     list at its innermost hit, in the head piece's frame (R22's passes; at a change
 *                                     of piece the state is rotated into the new frame, at a change of side zRef is
 *                                     re-based on the first hit of the new side and ndf loses 1); a chain of one piece
 *                                     keeps its tpc_fit_tracks result; chi2 = ndf = -1 if a transport ran into max_sinphi
 * K = counters[TPC_CNT_TRACKS] is read on the device.  Enqueue only.  TPC_EINVAL for missing buffers or parameters
 * out of range (chi2_cut, dz_max > 0, ce_tol >= 0, 1 <= max_rows <= 151, max_tracks <= 2^28), TPC_ENOMEM_WS for a short
 * workspace.
 * params->n_fit_passes must be even (TPC_EINVAL otherwise): the matching and the chain refit take the state of every
 * sector-local track at its INNERMOST hit, which is where tpc_fit_tracks leaves it after an even number of passes
 * (outward, inward, ...; the default is 2); after an odd number it sits at the outermost hit. */
typedef struct {
  float chi2_cut;    /* 50  */
  float dz_max;      /* 64 cm */
  float ce_tol;      /* 1 cm */
  int32_t max_rows;  /* 12 */
} tpc_merge_params_t;

typedef struct {
  int32_t* trk_succ;
  int32_t* trk_pred;
  float* trk_succ_chi2;
  int32_t* trk_global;
  int32_t* n_global;
  int32_t* g_head;
  int32_t* g_nseg;
  int32_t* g_nhits;
  float* gpar;
  float* gcov;
  float* gxref;
  float* gzref;
  float* gchi2;
  int32_t* gndf;
} tpc_merged_t;

int tpc_merge_workspace_bytes(const tpc_params_t* params_host, int64_t max_tracks, size_t* bytes_host);
int tpc_merge_tracks(const tpc_params_t* params_host, const tpc_merge_params_t* merge_host, int64_t n_clusters,
                     int64_t max_tracklets, const void* find_workspace, size_t find_ws_bytes,
                     const int32_t* counters, int64_t max_tracks, const tpc_result_t* dev, void* merge_workspace,
                     size_t merge_ws_bytes, const tpc_merged_t* out, void* stream);

/* ---- measurement support (bench.py `roofline`, `gpu_launches`) --------------------------------
 * The library counts every kernel it launches, per kernel id, and can bracket each launch with a
 * cudaEvent pair recorded on the launching stream.  Host-side state, one driving thread per GPU
 * (PAPER.md l.72).  Event timing is off by default and costs nothing on the device when off.
 *   tpc_profile_enable(on)   : switch event timing on/off and drop pending records
 *   tpc_profile_kernels()    : number of kernel ids;  tpc_profile_name(id): its name (static storage)
 *   tpc_profile_collect(n_ids, ms_host[n_ids] or NULL, launches_host[n_ids] or NULL, reset):
 *       waits for the recorded events, writes the summed elapsed ms and the launch counts per
 *       kernel id since the last reset; reset != 0 clears both.  At most 8192 timed launches are
 *       kept between collects (later ones are counted but not timed). */
int tpc_profile_enable(int on);
int tpc_profile_kernels(void);
const char* tpc_profile_name(int kernel_id);
int tpc_profile_collect(int n_ids, double* ms_host, int64_t* launches_host, int reset);
/* The FP32 roof the alu-bound kernels are reported against ("measure an FMA-chain peak"): runs a
 * kernel of independent FFMA chains (8 per thread, 8 blocks of 256 threads per SM) four times on `stream`,
 * SYNCHRONISES, and writes the best rate of the last three in TFLOP/s (2 flop per FMA) to *tflops_host.
 * scratch_dev: >= 4 bytes of device memory (never written in practice). */
int tpc_fp32_peak(float* scratch_dev, double* tflops_host, void* stream);

#ifdef __cplusplus
}
#endif
#endif /* TPC_B200_H_ */

/*
 * pslmc.h — C ABI of libpslmc: phase-space-let (PSL) source sampling + Monte Carlo dose on one B200.
 *
 * The operations are those of Tian et al., "An Analytic Linear Accelerator Source Model for Monte
 * Carlo dose calculations. II", in the reading fixed by DESIGN.md:
 *   psl_build          PAPER.md:35-57  §2.1.1 (PSR→PSL conversion, Eq. 1-2; ring-sector lets),
 *                      PAPER.md:61-69  §2.1.2 (sampling areas), :75-80 S1-S2 (Eq. 3)
 *   psl_build_grid     PAPER.md:39-55  the paper's own Cartesian (Xbin, Ybin) lets, steps 1-4
 *   psl_set_direction_model  PAPER.md:94-116 S4-S5, Eq. 6-7 (Gaussian mixtures in (alpha, beta))
 *   mc_plan_allocate,
 *   mc_plan_dose       PAPER.md:76-80  Eq. 3 across the beams of a plan; :73-75 one dose grid for the whole plan
 *   mc_sample_debug    PAPER.md:82-92  S3 (Eq. 4-5), :94-116 S4-S5, jaw rejection :65/:92, set-up :173
 *   mc_dose            PAPER.md:118-120 §2.1.3 (iterated source kernel / transport kernel, M per
 *                      launch, type-major / energy-ascending order), :161 (cut-offs 50 keV / 200 keV)
 *                      mc_opts_t.com_*: the commissioning tally, §2.2.2
 *   mc_stats           PAPER.md:177-191 Table 1 (per-phase timing breakdown)
 *
 * Conventions
 *   - Plain C structs, `extern "C"`, no exceptions cross the boundary, no torch types.
 *   - Every pointer says HOST or DEVICE.  The caller owns every array it passes and keeps it alive
 *     for the duration of the call.  The library owns `psl_t` (host + device tables) until psl_free.
 *   - Units: cm, MeV, g/cm^3.  Beam frame: origin at the primary source, +z downstream, isocentre at
 *     (0,0,sad).  Phantom frame: pos_ph = iso + R * (pos_beam - (0,0,sad)), dir_ph = R * dir_beam.
 *   - All entry points return 0 on success or a negative MC_E_* code; mc_last_error() returns a
 *     thread-local message.  Outputs are unspecified after an error.
 *   - The library keeps NO process-global device state: every byte of device scratch is the caller's
 *     `workspace` (mc_workspace_bytes / mc_host_workspace_bytes; NULL or too small -> MC_E_WORKSPACE, nothing
 *     is allocated inside mc_dose), every stream is the caller's (`cuda_stream`, `aux_streams`), the only
 *     device memory the library owns are the read-only tables of a psl_t (allocated by psl_build on the
 *     device current at that time, freed by psl_free).  Two host threads may therefore run mc_dose at the
 *     same time on different workspaces and streams (same or different psl_t: a psl_t is read-only after
 *     psl_build / psl_set_direction_model); a psl_t must be used on the device it was built on.
 *     mc_dose is synchronous with respect to the given stream when it returns.
 *   - Determinism: for fixed inputs and seed, dose, ledgers and counters are bitwise identical for
 *     every `batch`, every `order`, every `pipelines` and every partition [history_begin,history_end) summed.
 *   - There is no CPU fallback: every entry point that computes needs a CUDA device (sm_100a).
 */
#ifndef PSLMC_H
#define PSLMC_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define MC_OK             0
#define MC_E_INVALID_ARG -1
#define MC_E_EMPTY_FIELD -2  /* no let survives the jaw selection                              */
#define MC_E_WORKSPACE   -3  /* caller-supplied workspace too small                            */
#define MC_E_CUDA        -4  /* a CUDA runtime call or kernel failed                           */
#define MC_E_OVERFLOW    -5  /* the electron queue was full, or a voxel's int64 accumulator wrapped */

/* PSR analytic source model (paper layer L0).                           */
typedef struct {
  int32_t n_ebin, n_ring;          /* energy bins, rings                                         */
  double  e_min, e_bin_width;      /* MeV; bin e spans e_min + e*w .. e_min + (e+1)*w            */
  double  ring_width, z_phsp;      /* cm; ring i spans i*w .. (i+1)*w on the plane z = z_phsp    */
  const double *W;                 /* HOST [3][n_ebin][n_ring] relative ring weights, row-major  */
  double  sigma_src[3], z_src[3];  /* per sub-source Gaussian virtual source: sigma, plane z (cm)*/
  int32_t particle_type[3];        /* 0 photon, 1 electron                                       */
} psr_params_t;

/* Thin rectangular jaws.  Edges are given by their projection on the isocentre
 * plane z = sad; the X pair sits at z_jx, the Y pair at z_jy (beam frame, cm).  x1 < x2, y1 < y2. */
typedef struct { double x1, x2, y1, y2; double z_jx, z_jy, sad; } jaws_t;

/* Voxel phantom.  Voxel (i,j,k) spans o + i*d .. o + (i+1)*d per axis; linear index
 * (k*ny + j)*nx + i (x fastest).  Outside the grid is vacuum.                                   */
typedef struct {
  int32_t nx, ny, nz;
  double  dx, dy, dz, ox, oy, oz;
  const float   *density;          /* DEVICE (mc_dose) / HOST (mc_dose_host); g/cm^3             */
  const uint8_t *material;         /* DEVICE / HOST likewise; 0 water, 1 lung, 2 bone            */
} phantom_t;

/* Beam set-up ("translating and rotating").  R is row-major 3x3.                   */
typedef struct { double iso[3]; double R[9]; double sad; } beam_geom_t;

typedef struct psl psl_t;          /* opaque: active lets, alias tables, group weights           */

#define MC_ORDER_SORTED 0          /* sub-source major, energy bin ascending  */
#define MC_ORDER_MIXED  1          /* histories permuted, one combined launch over mixed types   */

#define MC_FLAG_ELECTRONS_LOCAL 1  /* debug physics: deposit every charged secondary on the spot */
#define MC_FLAG_STATS           2  /* fill the event counters of mc_stats_t (ledgers are always) */
#define MC_FLAG_TIMING          4  /* CUDA-event time per kernel class into mc_stats_t           */
#define MC_FLAG_STATIC_LANES    8  /* ablation: one particle per thread, no lane refill          */
#define MC_FLAG_STAGE_SCORING  16  /* stage the scoring atomics of hot voxels in shared memory    */
                                   /* (per-CTA table, added to the grid at kernel exit; same bits)  */
#define MC_FLAG_RANGE          32  /* take [history_begin, history_end) literally: [0, 0) is then   */
                                   /* the EMPTY range (a shard without work) instead of "everything" */
#define MC_FLAG_NO_TILE_SORT   64  /* overrides MC_FLAG_TILE_SORT                                   */
#define MC_FLAG_TILE_SORT     128  /* ablation: order every batch's particles by the tile of the     */
                                   /* phantom they enter (PAPER.md:118-120 spatial loop); same bits   */
#define MC_FLAG_FP_VOXELS     256  /* strict fingerprints: also the voxel of every deposit, the stream  */
                                   /* position after every accepted Kahn sampling and whether an electron */
                                   /* sub-step ended its condensed step (equal = same draws in the same roles) */

typedef struct {
  void     *workspace;             /* DEVICE scratch, REQUIRED: >= mc_workspace_bytes(psl, ph, batch)  */
  size_t    workspace_bytes;       /* (mc_dose_host: >= mc_host_workspace_bytes).  Contents are scratch. */
  void     *cuda_stream;           /* cudaStream_t or NULL (legacy default stream)               */
  int64_t  *dose_acc;              /* DEVICE int64[nx*ny*nz] or NULL.  When given, deposits are  */
                                   /* ADDED to it (multi-beam plans) and dose_out may be NULL    */
  int32_t   order;                 /* MC_ORDER_*                                                 */
  int32_t   flags;                 /* MC_FLAG_* bits                                             */
  uint64_t *fingerprints;          /* DEVICE u64[history_end-history_begin] or NULL; ADDED to    */
  uint64_t  history_begin;         /* sub-range of history ids to run (sharding) ...             */
  uint64_t  history_end;           /* ... 0 means n_histories (unless MC_FLAG_RANGE)             */
  int32_t   pipelines;             /* 0 = the default (3 when both aux_streams are given), 1 =      */
                                   /* strictly serial launches on cuda_stream (per-kernel times in    */
                                   /* mc_stats are then disjoint), at most 3.  With n > 1, batches    */
                                   /* are dealt round-robin to n launch sequences - on aux_streams[0], */
                                   /* aux_streams[1] and, the third, cuda_stream itself - so that one */
                                   /* kernel's tail overlaps another sequence's next kernel.  Same    */
                                   /* bits for every n.                                               */
  int32_t   reserved;              /* must be 0                                                    */
  /* commissioning tally, off when com_index is NULL: every history carries the */
  /* column of the PSR it was sampled from (its descendants inherit it): (stype*n_ebin+ebin)*n_ring */
  /* + ring for the photon sub-sources, 2*n_ebin*n_ring + ebin for electrons; a deposit in a voxel */
  /* with com_index[v] = 1 + row > 0 is also ADDED to com_dose[col * com_rows + row].              */
  const int32_t *com_index;        /* DEVICE int32[nx*ny*nz]                                       */
  int64_t  *com_dose;              /* DEVICE int64[com_cols * com_rows], quanta of 2^-32 MeV       */
  int32_t   com_rows, com_cols;    /* com_cols must be 2*n_ebin*n_ring + n_ebin; needs particle_type = {0,0,1} */
  /* streams of the pipelines (caller-owned cudaStream_t, e.g. torch streams; distinct from each other and from */
  /* cuda_stream).  The library forks them from cuda_stream and joins them back with events; NULL = serial.       */
  void     *aux_streams[2];
  /* mc_plan_dose only: this call runs shard `shard_index` of `shard_count` equal contiguous parts of EVERY beam's */
  /* history range (multi-GPU: one shard per rank, then one int64 all-reduce of dose_acc).  0, 0 = everything.      */
  int32_t   shard_index, shard_count;
  uint32_t  debug_eq_cap;          /* test hook: electron-queue capacity in entries (0 = the default 4*batch);   */
                                   /* the workspace layout keeps its full size.  Exercises MC_E_OVERFLOW.        */
  uint32_t  reserved2;             /* must be 0                                                    */
} mc_opts_t;

/* Ledger / kernel-class indices of mc_stats_t.                                                  */
enum { MC_LEDGER_INCIDENT = 0, MC_LEDGER_DEPOSITED = 1, MC_LEDGER_ESCAPED = 2, MC_LEDGER_JAW = 3 };
enum { MC_K_SAMPLE = 0, MC_K_PHOTON = 1, MC_K_ELECTRON = 2, MC_K_FINALISE = 3, MC_K_AUX = 4 };

typedef struct {
  /* energy ledgers in quanta of 2^-32 MeV, exact 128-bit sums as (hi:int64, lo:uint64)          */
  int64_t  ledger_hi[4];
  uint64_t ledger_lo[4];
  uint64_t n_hist[3];              /* histories sampled per sub-source                           */
  uint64_t n_jaw_rejected;
  /* event counters (MC_FLAG_STATS)                                                              */
  uint64_t n_missed;               /* tracks that never entered the phantom                      */
  uint64_t n_flights, n_virtual, n_compton, n_photo, n_pair;
  uint64_t n_photon_cutoff, n_photon_escape, n_uncollided_escape;
  uint64_t n_sec_electrons, n_sec_photons;
  uint64_t n_electron_tracks, n_electron_steps, n_electron_escape;
  uint64_t n_deposits;
  uint64_t n_kahn_trials;          /* Kahn rejection trials (accepted + rejected)                */
  uint64_t n_deflections;          /* multiple-scattering deflections = completed condensed steps */
  uint64_t queue_high_water;       /* electron queue, entries (the only queue: annihilation       */
                                   /* photons stay in the lane that converted)                     */
  uint64_t launches[5];            /* per MC_K_* class                                           */
  float    ms[5];                  /* per MC_K_* class (MC_FLAG_TIMING); with pipelines > 1 the    */
                                   /* classes overlap in time and their sum exceeds ms_total       */
  float    ms_total;               /* whole mc_dose on its stream, CUDA events (always)          */
} mc_stats_t;

/* psl_build — host.  Cuts every ring into n_sectors equal angular lets (weight W_ring/n_sectors,
 * Eq. 1-2 integrated over a sector), computes the sampling rectangle of each sub-source
 * (PAPER.md:65), keeps lets whose bounding box touches it, builds one alias table per
 * (sub-source, energy bin) group and uploads the tables to the current CUDA device.
 * Returns MC_E_EMPTY_FIELD if no let is active.                                                 */
int  psl_build(const psr_params_t *psr, const jaws_t *jaws, int32_t n_sectors, psl_t **out);
/* psl_build_grid — host.  The paper's own let shape (steps 1-4): a Cartesian grid of square
 * lets of side let_size (cm) over the phase-space disc, 2*ceil(r_max/let_size) lets per side (no let centre on
 * the axis).  Let weight = ring weight linearly interpolated along the radius at the let centre (between ring
 * centres; towards (0, 0) inside the first centre, constant beyond the last), divided by 2 pi r, normalised over all lets of all
 * energies and sub-sources.  A let is active when any portion of its square lies in the sampling rectangle of
 * its sub-source.  Everything else (alias tables, allocation, mc_dose) is as for psl_build; psl_export then
 * reports Xbin in ring[] and Ybin in sector[].                                                    */
int  psl_build_grid(const psr_params_t *psr, const jaws_t *jaws, double let_size, psl_t **out);
/* psl_set_direction_model — host.  Replaces the focal-geometry direction model of one sub-source by the paper's
 * Eq. 6 (scattered photons: K Gaussians in alpha = atan(u/w), beta = atan(v/w) per (energy bin, ring))
 * or Eq. 7 (electrons: K = 1, mu = 0).  c, mu, sigma_a, sigma_b: HOST double[n_ebin][n_ring][K]
 * (component weights, means of alpha, standard deviations; beta has mean 0).  The cumulative table
 * P_{i,k} = sum_{j<=k} c / sum_{j<=K} c is searched sequentially; (u, v) are local (u radial) and rotated by
 * atan2(y, x); the jaw test is done on the ray from the phase-space point.  K = 0 restores the focal model.
 * K <= 8.  Uploads the table to the current device.                                                      */
int  psl_set_direction_model(psl_t *psl, int32_t stype, int32_t K, const double *c, const double *mu,
                             const double *sigma_a, const double *sigma_b);
void psl_free(psl_t *psl);

/* psl_export — host.  Serialises the tables for inspection:
 *   u64 n_groups; then per group: i32 stype, i32 ebin, u64 n, f64 W_g,
 *   u16 ring[n], u16 sector[n], u32 thresh[n], u32 alias[n]   (each array padded to 8 bytes);
 *   finally f64 rect[3][4] = (xlo,xhi,ylo,yhi) sampling rectangle per sub-source.
 * Call with host_buf = NULL to get the size in *bytes.                                          */
int  psl_export(const psl_t *psl, void *host_buf, size_t *bytes);

/* psl_allocate — host.  Eq. 3 at group level: N_g = N*W_g/sum(W_g), largest-remainder rounding.
 * off_out: HOST u64[n_groups+1], prefix offsets of the contiguous history-id ranges.            */
int  psl_allocate(const psl_t *psl, uint64_t n_histories, uint64_t *off_out);

/* mc_plan_allocate — host.  Eq. 3 across the beams of a treatment plan (the denominator of Eq. 3 runs
 * over the sampling areas of all beams): beam i gets n_histories * W_i / sum_j W_j histories, W_i = the sum of the
 * active group weights of psls[i]; largest-remainder rounding, ties to the lower index.  n_out: HOST u64[n_beams].
 * Run mc_dose once per beam with n_out[i] histories into one opts->dose_acc, then scale by the plan total.      */
int  mc_plan_allocate(const psl_t *const *psls, int32_t n_beams, uint64_t n_histories, uint64_t *n_out);

/* Workspace bytes mc_dose / mc_plan_dose / mc_transport_debug need for this batch size (0 on invalid arguments;
 * psl may be NULL: the layout depends on the phantom's voxel count and the batch only).                        */
size_t mc_workspace_bytes(const psl_t *psl, const phantom_t *ph, uint64_t batch);
/* The same plus the device staging of mc_dose_host (phantom arrays in, dose out: 13 bytes per voxel).          */
size_t mc_host_workspace_bytes(const psl_t *psl, const phantom_t *ph, uint64_t batch);

/* mc_dose — the hot path.  Runs histories [history_begin,history_end) of an n_histories-history
 * allocation in batches of `batch` through k_sample → k_photon / k_electron (+ secondary queues)
 * with int64 fixed-point scoring, then writes
 *   dose_out[v] = acc[v] * 2^-32 / (rho_v * V_voxel * n_histories)   (MeV/g per history; 0 if rho=0)
 * dose_out: DEVICE double[nx*ny*nz], overwritten (may be NULL if opts->dose_acc is given).      */
int  mc_dose(const psl_t *psl, const phantom_t *ph, const beam_geom_t *beam,
             uint64_t n_histories, uint64_t seed, uint64_t batch,
             double *dose_out, const mc_opts_t *opts);

/* mc_dose_static — mc_dose for callers that may not allocate device memory (code whose surroundings are under CUDA
 * graph capture, serving loops, harnesses that forbid cudaMalloc).  Same arguments, same kernels, same bits as mc_dose,
 * except that opts->workspace / workspace_bytes must be NULL / 0: the scratch is a file-scope `static __device__` array
 * of MC_STATIC_WORKSPACE_BYTES inside the library (every GPU that loads libpslmc holds it until the process exits; its
 * device address is taken once per device with cudaGetSymbolAddress on the device current at the first call).  Needs
 * mc_workspace_bytes(psl, ph, batch) <= MC_STATIC_WORKSPACE_BYTES, else MC_E_WORKSPACE (nothing is launched): e.g. a
 * 64^3 phantom with batch <= 2^16, or a 128^3 phantom with batch <= 2^15.  The call itself and everything below it
 * calls no cudaMalloc, cudaFree or other allocating routine (it creates and destroys CUDA events, like mc_dose).
 * The array is shared by every call on that device and keeps the last call's contents; the call clears what must start
 * at zero.  Two mc_dose_static calls that overlap on one GPU (different streams or host threads) RACE on it: serialise
 * them, or give the others their own workspace through mc_dose.  Inputs and outputs stay the caller's.                */
#define MC_STATIC_WORKSPACE_BYTES (64u << 20)
size_t mc_static_workspace_bytes(void);
int  mc_dose_static(const psl_t *psl, const phantom_t *ph, const beam_geom_t *beam,
                    uint64_t n_histories, uint64_t seed, uint64_t batch,
                    double *dose_out, const mc_opts_t *opts);

/* mc_dose_host — same, end to end from HOST buffers: ph->density / ph->material and dose_out are
 * HOST pointers (pinned memory makes the copies asynchronous); the call uploads the phantom into the
 * workspace, runs mc_dose, and downloads the dose.  opts->workspace >= mc_host_workspace_bytes.  */
int  mc_dose_host(const psl_t *psl, const phantom_t *ph_host, const beam_geom_t *beam,
                  uint64_t n_histories, uint64_t seed, uint64_t batch,
                  double *dose_out_host, const mc_opts_t *opts);

/* mc_plan_dose — a treatment plan of n_beams beams on one phantom (PAPER.md:73-80 S1-S2): Eq. 3 over the sampling
 * areas of ALL beams gives beam i its n_i of the plan's n_histories (mc_plan_allocate); beam i then runs exactly
 * like mc_dose(psls[i], ph, &beams[i], n_i, seed + i, batch) and every beam scores into ONE int64 grid
 * (opts->dose_acc when given - deposits are ADDED - else a grid inside the workspace, zeroed first).
 *   dose_out[v] = acc[v] * 2^-32 / (rho_v * V_voxel * n_histories)     (DEVICE double[nvox] or NULL)
 * opts->shard_index / shard_count select one of shard_count equal contiguous parts of every beam's history range;
 * the shards' int64 grids add up bit for bit to the unsharded plan.  history_begin/end, fingerprints, order and
 * the commissioning tally are not available at plan level (MC_E_INVALID_ARG).  n_beam_out: HOST u64[n_beams] or NULL.
 * mc_stats afterwards holds the sums over the beams (ledgers, counters, launches, milliseconds).                  */
int  mc_plan_dose(const psl_t *const *psls, const beam_geom_t *beams, int32_t n_beams, const phantom_t *ph,
                  uint64_t n_histories, uint64_t seed, uint64_t batch, double *dose_out, const mc_opts_t *opts,
                  uint64_t *n_beam_out);

/* Counters, ledgers and timings of the last mc_dose / mc_plan_dose / mc_transport_debug on this thread. */
int  mc_stats(mc_stats_t *out);
const char *mc_last_error(void);

/* ---- parity / debug exports ------------------------------------------------------------------ */

/* Source sampling only.  soa_out: DEVICE float[8*count] as two float4 planes,
 *   plane 0 [i] = (x, y, z, E), plane 1 [i] = (u, v, w, status), i = history - first_history,
 * status = group index (>= 0) if the particle passed the jaws, -(group index) - 1 if rejected.  */
int  mc_sample_debug(const psl_t *psl, const beam_geom_t *beam, uint64_t first_history,
                     uint64_t count, uint64_t n_histories, uint64_t seed, float *soa_out,
                     void *cuda_stream);

/* Transport only.  Takes `count` particles in the layout of mc_sample_debug (status < 0 entries
 * are skipped), particle_type 0 photon / 1 electron, as track 0 of histories first_history + i
 * with the stream positioned at block 2, and scores into opts->dose_acc (required).  Ledgers and
 * counters go to mc_stats; the incident ledger counts the particles given.                      */
int  mc_transport_debug(const phantom_t *ph, int32_t particle_type, const float *soa_in,
                        uint64_t first_history, uint64_t count, uint64_t seed,
                        const mc_opts_t *opts);

/* The photon cross-section lookup of k_photon (per-call table in log2 E, linear interpolation) for a
 * list of energies: builds the table for the given largest density per material (rhomax[3]: water,
 * lung, bone) and top energy e_max (MeV, > 0.05), then evaluates it ON THE DEVICE.
 * E_host: HOST float[n] (0.05 <= E <= e_max); out_host: HOST float[3n] = (sigma_KN cm^2 per electron,
 * ln^2(E/1.022) or 0 below threshold, mu_max cm^-1) per energy.                                  */
int  mc_xs_debug(const float rhomax[3], double e_max, const float *E_host, uint64_t n, float *out_host);

/* One Philox4x32-10 block computed ON THE DEVICE: key = seed, counter = (block, track, h_lo, h_hi).
 * out: HOST u32[4].                                                                             */
int  mc_philox_debug(uint64_t seed, uint64_t history, uint32_t track, uint32_t block,
                     uint32_t *out);

#ifdef __cplusplus
}
#endif
#endif /* PSLMC_H */

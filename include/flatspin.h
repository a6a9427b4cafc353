/* flatspin.h -- C ABI of the B200-native flatspin hot path (libflatspin_b200.so).
 *
 * What it computes is defined by /root/reference/PAPER.md (arxiv 2002.11401, "flatspin: A Large-Scale
 * Artificial Spin Ice Simulator"); citations below are PAPER.md lines.  SURVEY.md section 8(b) lists
 * the entry points.  No torch types cross this boundary: plain pointers (each marked DEVICE or HOST)
 * and sizes.  All kernels are hand-written CUDA for sm_100a (paper_2002_11401_b200/csrc/flatspin.cu).
 *
 * Model (Eq. 1): N binary macro spins s_i in {-1,+1} at positions r_i with rotation
 * theta_i and coercive field h_c^(i) (== h_k^(i) of Eq. 5, reading C-4).
 *
 * Conventions
 *   - Every DEVICE pointer is caller-owned CUDA global memory (a torch tensor's data_ptr()).  Inputs
 *     of fs_create* are consumed during the call and may be freed afterwards.  The workspace is
 *     caller-owned and must outlive the handle.  Outputs are written to caller-owned buffers.
 *     The workspace holds every per-spin and per-interaction array, the flip log, the batched-flip scratch (35 MB at
 *     config 4) and the per-spin external field of fs_set_local_field.  The one thing the library allocates itself
 *     (cudaMalloc in fs_create, freed by fs_destroy, NOT counted by fs_workspace_bytes) is the lattice-stencil table set,
 *     whose size is known only after the lattice detection: index grids and dense spin grids of <= 8N + 2^20 cells per
 *     replica, a cell index (4N bytes) and a few KB of couplings (30 MB at config 5); none when the geometry is not a
 *     lattice.  Temporaries of fs_workspace_bytes / fs_create (detection scratch, 9N bytes) / fs_measure_*_peak are
 *     freed before the call returns.
 *     fs_scan_static (below) is the one entry point that touches no allocator at all.
 *   - HOST pointers to scalars (n_flips_out ...) are written after a stream synchronise; passing NULL
 *     skips the synchronise (the call is then fully asynchronous on `stream`).
 *   - All work is enqueued on the stream given at creation (a cudaStream_t passed as void*; NULL =
 *     the legacy default stream).
 *   - Fields are (parallel, perpendicular) pairs in the FIXED geometric frame of theta_i:
 *       par = h . (cos theta_i, sin theta_i),  perp = h . (-sin theta_i, cos theta_i)
 *     (Fig. 2; reading C-2).  Eq. 6 then reads s_i * par < 0.
 *   - Ensembles: R independent replicas share the geometry and differ in h_c, spins
 *     and thermal seed (seed + r).  Arrays carry a leading [R] dimension.  R == 1 for fs_create.
 *   - Return value: FS_OK (0) or a negative FS_ERR_* code; fs_last_error() gives a message for the
 *     calling thread.  No exception crosses the ABI.  There is NO CPU fallback: without a CUDA
 *     device every compute entry point returns FS_ERR_CUDA.
 */
#ifndef FLATSPIN_B200_H
#define FLATSPIN_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct fs_sim fs_sim; /* opaque; owned by the library; freed by fs_destroy */

/* alpha: dipolar coupling strength (Eq. 3).  b, c, beta, gamma: generalized
 * Stoner-Wohlfarth astroid (Eq. 5).  neighbor_distance: neighbourhood radius in
 * lattice units; j is a neighbour of i iff j != i and |r_i-r_j|^2 <= nd^2 (1+1e-9)
 * (reading A-7). */
typedef struct {
    double alpha, b, c, beta, gamma, neighbor_distance;
} fs_params;

enum {
    FS_OK = 0,
    FS_ERR_ARG = -1,        /* null pointer, N<=0, R<=0, hc<=0 or non-finite, b,c,beta,gamma,nd <= 0, K too large */
    FS_ERR_COINCIDENT = -2, /* two distinct spins at the same position (Eq. 3 singular; reading C-8) */
    FS_ERR_WORKSPACE = -3,  /* workspace too small or misaligned (needs 256-byte alignment) */
    FS_ERR_CUDA = -4,       /* CUDA runtime error, or no device */
    FS_ERR_MAXFLIPS = -5    /* fs_relax stopped at max_flips with switchable spins left; state valid */
};

/* Which field fs_get_fields returns (Eq. 2): h_i = h_dip + h_ext + h_th. */
enum { FS_FIELD_TOTAL = 0, FS_FIELD_DIP = 1, FS_FIELD_EXT = 2, FS_FIELD_THERMAL = 3 };

/* Gather kernel variants for fs_update_fields:
 *   0 = auto: the lattice stencil when the geometry was detected to be a regular lattice, else ELL;
 *   1 = ELL: neighbour indices + fp64 coupling pairs streamed from HBM (20 B / interaction; HBM-bound);
 *   2 = lattice stencil: dense per-sublattice spin grids correlated with the table
 *       T[sub_i][sub_j][du][dv] = alpha*g_ij held in shared memory (no per-interaction HBM traffic;
 *       FP64-pipe bound).  FS_ERR_ARG if the geometry is not a verified regular lattice.  Where the table has an
 *       exact inversion pairing (Eq. 3 is even in r_ij: T[d] == T[-d], bit for bit) the kernel adds the two
 *       spins of a slot pair first: 3 FP64 operations per 2 interactions instead of 4;
 *   3 = lattice stencil without the inversion pairing (one DFMA pair per interaction);
 *   4 = the OPTIONAL fp32 field path (BASELINE.json north_star: "reported separately at 1e-5"): the same stencil
 *       kernel in single precision (couplings rounded to fp32, fp32 accumulation), h_dip stored as double.  Fields
 *       agree with the fp64 paths to ~1e-6 relative to max|h|; spin / flip-order parity is NOT claimed after it (the
 *       decision gaps of the relaxation are far below fp32 resolution).  Never chosen automatically.  FS_ERR_ARG unless
 *       the geometry is a verified lattice whose table fits constant memory. */
enum { FS_GATHER_AUTO = 0, FS_GATHER_ELL_F64 = 1, FS_GATHER_STENCIL = 2, FS_GATHER_STENCIL_PLAIN = 3, FS_GATHER_STENCIL_F32 = 4 };

/* Why the stencil is not available (fs_get_lattice info[1]); 0 = it is. */
enum {
    FS_LATTICE_OK = 0,
    FS_LATTICE_NO_NEIGHBORS = 1,          /* K == 0: nothing to gather */
    FS_LATTICE_NO_BASIS = 2,              /* no two lattice vectors found around the reference spin */
    FS_LATTICE_TOO_MANY_SUBLATTICES = 3,  /* more than 8 */
    FS_LATTICE_NOT_PERIODIC = 4,          /* spins off the lattice, or two spins in one cell */
    FS_LATTICE_STENCIL_TOO_WIDE = 5,      /* half-extent > 40 cells or shared memory exceeded */
    FS_LATTICE_TOO_SPARSE = 6,            /* dense grids would exceed 8N + 2^20 cells */
    FS_LATTICE_REACH_MISMATCH = 7,        /* stencil would reach a different set of pairs than the ELL */
    FS_LATTICE_WEIGHT_MISMATCH = 8        /* couplings of equal offsets differ by more than 5e-13/K relative to max|w| */
};

/* Bytes of workspace fs_create[_ensemble] needs for this geometry (runs the cell-grid neighbour count,
 * PAPER.md:57, to find the maximum degree K).  pos_dev: DEVICE [N,2] row-major fp64.
 * bytes_out: HOST.  Synchronises `stream`. */
int fs_workspace_bytes(int64_t N, int32_t R, const double* pos_dev, const fs_params* p,
                       size_t* bytes_out, void* stream);

/* Build a simulation: frame tables (Eq. 1), cell-grid neighbour lists, couplings
 * alpha*g_ij (Eq. 3) in row-major ELL.  Spins start at +1 (fs_set_spins to change).
 * pos_dev DEVICE [N,2]; angle_dev DEVICE [N] radians; hc_dev DEVICE [N] (fs_create) or [R,N]
 * (fs_create_ensemble), all > 0.  workspace_dev: DEVICE, 256-byte aligned, >= fs_workspace_bytes.
 * Synchronises `stream` once (to read K and the validation flags).  N <= 16,777,216 spins per replica (the relax
 * loop keeps up to 16,384 leaf maxima of up to 1024 spins in shared memory): FS_ERR_ARG beyond. */
int fs_create(fs_sim** out, int64_t N, const double* pos_dev, const double* angle_dev,
              const double* hc_dev, const fs_params* p, void* workspace_dev, size_t workspace_bytes,
              void* stream);
int fs_create_ensemble(fs_sim** out, int64_t N, int32_t R, const double* pos_dev,
                       const double* angle_dev, const double* hc_dev, const fs_params* p,
                       void* workspace_dev, size_t workspace_bytes, void* stream);
int fs_destroy(fs_sim* sim);

/* Geometry queries (HOST outputs, no synchronise). */
int fs_get_info(const fs_sim* sim, int64_t* N, int32_t* R, int32_t* K /*max degree*/,
                int64_t* n_interactions /*sum of degrees*/);

/* s_dev: DEVICE [R,N] int8, values +1/-1.  Marks h_dip stale (recomputed lazily by the next call
 * that needs it, or explicitly by fs_update_fields). */
int fs_set_spins(fs_sim* sim, const int8_t* s_dev);
int fs_get_spins(fs_sim* sim, int8_t* s_dev_out /*DEVICE [R,N]*/);

/* Thermal field: per spin and step two components sigma_th * N(0,1) in global x,y from
 * Philox4x32-10 keyed (seed + replica; step; spin) + Box-Muller (reading C-11), constant
 * during a relaxation.  sigma_th = 0 switches it off (default). */
int fs_set_thermal(fs_sim* sim, double sigma_th, uint64_t seed);

/* Global external field for all replicas, and the step key of the thermal stream.  Host values; no launch
 * and no synchronise: the next scan / relax takes the field as a kernel argument.  Always FS_OK for a valid sim. */
int fs_set_field(fs_sim* sim, double hx, double hy, uint32_t step);
/* Per-replica global fields: h_host HOST [R,2] (hx,hy). */
int fs_set_field_ensemble(fs_sim* sim, const double* h_host, uint32_t step);

/* Per-spin external field h_ext^(i) ("global, per-spin or a spatial vector field"): h_dev DEVICE
 * [N,2] (global x,y components), shared by all replicas, ADDED to the global field of fs_set_field / fs_sweep
 * before the rotation into the spin's frame (reading D-4).  Copied (into the workspace); NULL
 * clears it.  Takes effect at the next scan / relax / sweep. */
int fs_set_local_field(fs_sim* sim, const double* h_dev);

/* Choose the gather kernel variant (FS_GATHER_*).  Default auto. */
int fs_set_gather_variant(fs_sim* sim, int variant);

/* Result of the regular-lattice detection run by fs_create (flatspin geometries are
 * lattices with 1-3 sublattices, :146).  info HOST [12] int32: {stencil active, FS_LATTICE_* reason,
 * sublattices, U, V (cells along the two lattice vectors), Ru, Rv (stencil half-extents), stencil
 * slots present, warps per CTA, shared-memory bytes per CTA, inversion pairing active, row pairs}.  dinfo HOST [2]: {max |w_ELL - T| over
 * all interactions, max |w|}.  Either may be NULL.  No synchronise. */
int fs_get_lattice(const fs_sim* sim, int32_t* info, double* dinfo);

/* Calibration for the FP64 roofline: runs a chain of dependent-free DFMAs on every SM and
 * returns the best of 4 timed launches in DFMA/s (HOST).  Synchronises `stream`. */
int fs_measure_fp64_peak(double* dfma_per_s, void* stream);
/* The same for fp32 FFMA/s (denominator of the optional fp32 field path's roofline). */
int fs_measure_fp32_peak(double* ffma_per_s, void* stream);

/* Full dipolar-field gather h_dip,i = sum_k s[nbr[i][k]] * w[i][k] for every spin (Eq. 3 over the
 * neighbourhood).  Asynchronous. */
int fs_update_fields(fs_sim* sim);

/* Fused total field + astroid + switching margin + arg-max (Eqs. 2, 5, 6), replica 0
 * of an ensemble unless *_ensemble.  Outputs HOST: number of switchable spins, the index of the
 * spin furthest outside its astroid (lowest index among exact ties; -1 if none) and its Eq. 5
 * left-hand side.  Synchronises. */
int fs_scan(fs_sim* sim, int64_t* n_switchable, int64_t* best_index, double* best_L);
int fs_scan_ensemble(fs_sim* sim, int64_t* n_switchable /*HOST [R]*/, int64_t* best_index /*HOST [R]*/,
                     double* best_L /*HOST [R]*/);

/* Relaxation: repeat { flip the switchable spin with the greatest Eq. 5 left-hand
 * side; update its neighbours' h_dip incrementally } until no spin is switchable, entirely on the
 * device.  max_flips <= 0: unlimited.  n_flips_out HOST (sum over replicas for an ensemble; NULL =
 * asynchronous, read later with fs_get_counters).  Returns FS_ERR_MAXFLIPS if the cap stopped it
 * (only detected when n_flips_out != NULL). */
int fs_relax(fs_sim* sim, int64_t max_flips, int64_t* n_flips_out);
int fs_relax_ensemble(fs_sim* sim, int64_t max_flips, int64_t* n_flips_out /*HOST [R]*/);

/* Exact batched flips: for one large system (R = 1, 1 <= K <= 64, N >= 16384, no max_flips cap)
 * fs_relax first runs a kernel on all SMs that commits, per round, the longest prefix of the sequential flip
 * sequence of PAPER.md:122 (":129-130 switching is sequential") that it can prove exact: up to `max_seeds` top
 * candidates, joined into components where their closed neighbourhoods overlap, each relaxed locally by one warp,
 * merged by effective key, cut at the first conflict (batch.cuh has the argument).  The flip log, spins and fields
 * are identical to the one-flip-at-a-time loop, which still finishes the tail once fewer than `seq_threshold`
 * spins are switchable.  max_seeds = 0 switches the batched kernel off; the default is about 4 sqrt(N / (K+1)) (the
 * measured optimum: commits per round grow with the seeds, collisions between regions with their square), the
 * maximum twice that (at most 4096).
 * fs_get_batch_stats: out4 HOST [4] = {max_seeds in use (0 = off), flips committed by the batched kernel, its
 * rounds (mean committed prefix = flips / rounds), seq_threshold} since creation / the last counter reset.
 * Synchronises. */
int fs_set_batch(fs_sim* sim, int32_t max_seeds, int32_t seq_threshold);
int fs_get_batch_stats(fs_sim* sim, int64_t* out4);

/* A whole field protocol in ONE launch (PAPER.md:63 "discrete time series"; :124 relaxed at each value):
 * for t = 0..T-1 { global field fields[t]; thermal step key step0 + t; scan (Eqs. 2, 5, 6); relax
 * }, one persistent CTA per replica doing the scan itself, no host involvement between
 * steps.  Same arithmetic and flip order as T calls of fs_set_field + fs_relax.  Meant for small and
 * medium systems and for ensembles, where per-step launches dominate; for N >~ 10^5 the
 * multi-kernel path scans faster.  fields_dev DEVICE [T,2] (hx,hy), shared by all replicas;
 * flips_per_step_dev DEVICE [R,T] int64 or NULL; max_flips <= 0: unlimited (cap on the whole sweep);
 * n_flips_out HOST [R] (total flips of the sweep) or NULL = asynchronous.  The flip log
 * (fs_get_flip_log) then holds the flips of the whole sweep in order (the last 4N+1024 of them).
 * If the cap stops a replica inside the protocol (FS_ERR_MAXFLIPS, reported only with n_flips_out != NULL) its
 * state is that of the step it reached: the global field is fields[that step], flips_per_step of the steps
 * never run is 0, and the thermal step key used by fs_get_fields becomes step0 + (the step replica 0 reached). */
int fs_sweep(fs_sim* sim, const double* fields_dev, int32_t T, uint32_t step0, int64_t* flips_per_step_dev,
             int64_t max_flips, int64_t* n_flips_out);

/* fs_sweep with a thermal field strength per step: sigma_dev DEVICE [T] (annealing with an
 * exponentially decreasing thermal field); NULL = the constant sigma of fs_set_thermal.  The seed is the one
 * of fs_set_thermal; after the call fs_get_fields(THERMAL/TOTAL) still uses fs_set_thermal's sigma (call
 * fs_set_thermal with the last value to read the final thermal field). */
int fs_sweep_anneal(fs_sim* sim, const double* fields_dev, const double* sigma_dev, int32_t T, uint32_t step0,
                    int64_t* flips_per_step_dev, int64_t max_flips, int64_t* n_flips_out);

/* fs_sweep with time-dependent per-spin fields ("h_ext is a discrete time series of either local,
 * global or spatial fields"): at step t the external field of spin i is
 *     h_ext^(i)(t) = fields[t] + local_scale[t] * local_i + local_series[t][i]        (global x,y components)
 * local_i = the static per-spin field of fs_set_local_field (its scale defaults to 1), local_scale_dev DEVICE [T] or
 * NULL, local_series_dev DEVICE [T,N,2] or NULL (shared by all replicas), sigma_dev as fs_sweep_anneal.  Rounded as
 * written: (scale * local) + series, then added to the global field, then rotated (reading D-4).
 * After the call fs_get_fields(EXT/TOTAL) uses the static local field only. */
int fs_sweep_ex(fs_sim* sim, const double* fields_dev, const double* sigma_dev, const double* local_scale_dev,
                const double* local_series_dev, int32_t T, uint32_t step0, int64_t* flips_per_step_dev,
                int64_t max_flips, int64_t* n_flips_out);

/* Analysis reductions of the current spin state (PAPER.md:204-206 section IV.B; :160 "analysis of vertex populations").
 * fs_correlation: spin-spin correlation by separation.  c_ij = +1 (-1) if the dipole interaction of the pair is
 * minimised (maximised): sign of s_i s_j g_par,ij; pairs whose parallel coupling vanishes (|g_par| d^3 < 1e-9) are
 * skipped.  Every unordered pair of the neighbourhood once, bin = floor(|r_ij| / bin_width), pairs beyond nbins
 * (<= 2048) dropped.  sum_dev DEVICE [R,nbins] int64 = sum of c_ij per replica, count_dev DEVICE [nbins] int64 =
 * pairs per bin (geometry only); the correlation at a separation is sum / count (average over replicas for an
 * ensemble).  Asynchronous.
 * fs_vertex_populations: vertices_dev DEVICE [V,4] int32 = the four spins meeting at each vertex (square / pinwheel
 * ASI); counts_dev DEVICE [R,4] int64 = number of Type I, II, III, IV vertices: moments pointing into the vertex
 * 0 or 4 -> IV, 1 or 3 -> III, 2 -> I if they are opposite (zero net moment), II if adjacent. */
int fs_correlation(fs_sim* sim, double bin_width, int32_t nbins, int64_t* sum_dev, int64_t* count_dev);
int fs_vertex_populations(fs_sim* sim, const int32_t* vertices_dev, int64_t V, int64_t* counts_dev);

/* Counters accumulated on the device since creation / the last reset: HOST [R] each (any may be
 * NULL).  Synchronises. */
int fs_get_counters(fs_sim* sim, int64_t* total_flips, int64_t* last_relax_flips, int reset);

/* h_dev_out DEVICE [R,N,2] (par, perp) in the fixed theta_i frame; `which` = FS_FIELD_*. */
int fs_get_fields(fs_sim* sim, int which, double* h_dev_out);

/* Flip log of the last fs_relax / fs_sweep of replica `replica`: idx_dev_out DEVICE [cap] int32 in flip order;
 * n_out HOST = number of flips of that call.  The internal log is a ring of 4N+1024 entries: when a long sweep
 * (many field periods) makes more flips than that, the LAST 4N+1024 are kept.  The output starts at the oldest
 * flip still held, number *first_out (HOST, may be NULL; 0 unless the ring wrapped), and holds
 * min(cap, n - first) entries.  fs_get_flip_log is the same without first_out.  Synchronises. */
int fs_get_flip_log(fs_sim* sim, int32_t replica, int32_t* idx_dev_out, int64_t cap, int64_t* n_out);
int fs_get_flip_log_window(fs_sim* sim, int32_t replica, int32_t* idx_dev_out, int64_t cap, int64_t* n_out,
                           int64_t* first_out);

/* Neighbour table: idx_dev_out DEVICE [N,K] row-major int32, ascending, -1 padded; K_out HOST. */
int fs_get_neighbors(fs_sim* sim, int32_t* idx_dev_out, int32_t* K_out);

/* Host-buffer convenience for end-to-end timing: H2D spins [R,N] -> gather -> scan -> D2H total fields
 * [R,N,2], all on the simulation's stream, then synchronise.  s_host / h_host_out HOST (pinned for
 * full speed).  h_host_out may be NULL: then only the scan's summary returns to the host (the fields stay on the
 * device, as they do for fs_relax).  Scan outputs as fs_scan (replica 0). */
int fs_step_host(fs_sim* sim, const int8_t* s_host, double* h_host_out, int64_t* n_switchable,
                 int64_t* best_index, double* best_L);

/* Host-buffer relaxation step: set the field, relax, D2H spins [R,N].  n_flips_out HOST (sum). */
int fs_relax_host(fs_sim* sim, double hx, double hy, uint32_t step, int8_t* s_host_out,
                  int64_t* n_flips_out);

/* The switching scan for callers that must not allocate device memory (Eqs. 2, 5, 6 and the arg-max of PAPER.md:122;
 * SURVEY.md A4-A7).
 *
 * Every other scan here works on a handle whose partial results live in the workspace fs_create laid out.  Some callers
 * cannot provide one, and cannot let this library allocate either: a program whose own memory pool already holds
 * (nearly) all of the card (a torch caching allocator sized for config 5's workspace, a solver that reserves HBM at
 * start-up) would see a cudaMalloc inside the library fail or eat memory the pool counts on; a program that keeps
 * several streams busy would see every cudaMalloc / cudaFree synchronise the whole device.  fs_scan_static needs no
 * handle and no workspace and calls no cudaMalloc, cudaFree or other allocating routine: the per-CTA partial maxima
 * and the ticket counter of its arg-max live in a fixed array inside the library image, FS_SCAN_STATIC_SCRATCH_BYTES
 * per GPU that loads the library, held until the process exits.  That array bounds the size: N <= FS_SCAN_STATIC_MAX_N
 * (1024 spins per CTA, one 16-byte partial result each); larger N returns FS_ERR_ARG and launches nothing.
 *
 * Inputs, all DEVICE, caller-owned, read only: angle_dev [N] radians (Eq. 1), hc_dev [N] > 0 (h_k^(i) of Eq. 5),
 * s_dev [N] int8 +1/-1, hdip_dev [N,2] = (par, perp) of h_dip in the fixed frame of theta_i, 16-byte aligned (what
 * fs_get_fields(FS_FIELD_DIP) returns).  p: HOST; only b, c, beta, gamma are read.  (hx, hy): global external field;
 * sigma_th, seed, step: thermal field exactly as fs_set_thermal + fs_set_field define it (sigma_th = 0: none).
 * Output: result_dev DEVICE, 24 bytes, 8-byte aligned: { int64 number of switchable spins, int64 index of the spin
 * furthest outside its astroid (lowest index among exact ties; -1 if none), double its Eq. 5 left-hand side (-inf if
 * none) } -- the three values fs_scan returns for the same state, same arithmetic.  Asynchronous on `stream` (of the
 * CURRENT device, which must own all the pointers); no synchronise.
 *
 * First call on a device: looks up the array's device address (cudaGetSymbolAddress, which may load the library's
 * kernels on that device).  Make that first call outside any stream capture; later calls only enqueue a 256-byte
 * memset of the counter and one kernel.
 * Sharing: all calls on one device use the same array.  Calls on one stream, or otherwise ordered, are safe in any
 * number and any mix of sizes (the counter is cleared per call; stale partial results are never read).  Two calls that
 * can overlap on the GPU (different streams, no event between them) race on the array and give undefined results. */
#define FS_SCAN_STATIC_MAX_N 4194304
#define FS_SCAN_STATIC_SCRATCH_BYTES 65792 /* 256 (counter) + 16 * FS_SCAN_STATIC_MAX_N / 1024 */
int fs_scan_static(int64_t N, const double* angle_dev, const double* hc_dev, const int8_t* s_dev, const double* hdip_dev,
                   const fs_params* p, double hx, double hy, double sigma_th, uint64_t seed, uint32_t step,
                   void* result_dev, void* stream);

/* Number of kernels this library launched since load (all sims), for the benchmark's launch count. */
int64_t fs_kernel_launches(void);

const char* fs_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* FLATSPIN_B200_H */

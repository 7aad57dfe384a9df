/*
 * xy.h -- C-ABI boundary of the B200-native Swendsen-Wang sweep for the 2D classical XY model
 * (arXiv 1210.6116, Komura & Okabe).  Plain pointers and sizes only; nothing throws or aborts
 * across this boundary.  Every function returns XY_OK (0) or a negative XY_ERR_* code;
 * xy_last_error() returns a thread-local, human-readable message for the last failure.
 *
 * The model (Eq. 3): H = -J sum_<ij> cos(theta_i - theta_j) on an L x L square
 * lattice with periodic boundaries, J = 1.  Site index i = y*L + x (row-major);
 * site i owns its +x bond to R(i) = y*L + (x+1 mod L) and its +y bond to D(i) = ((y+1) mod L)*L + x.
 *
 * One sweep (the hot path; Swendsen-Wang multi-cluster update PAPER.md:22 with Wolff's embedded
 * cluster formalism PAPER.md:26; formulas as fixed in DESIGN.md section 3):
 *   1. direction  phi_t uniform on [0, 2pi), r = (cos phi, sin phi)
 *   2. projection sigma_i = s_i . r = cos(theta_i - phi)
 *   3. bonds      bond <ij> active iff u < 1 - exp(-2 beta sigma_i sigma_j)   (decision in fp64)
 *   4. labels     connected components of the active bonds; label = minimum site index
 *   5. flip       each cluster reflected theta -> 2 phi + pi - theta (mod 2pi) with probability 1/2
 *   6. observe    E, M, and the helicity-modulus link sums of Eq. 4-6
 * All random numbers come from Philox4x32-10 keyed by (seed; index, sweep counter t, tag), so a
 * sweep is a deterministic function of (theta, seed, t, beta).
 *
 * Threading / devices: a state is bound to the CUDA device current at creation and is not
 * thread-safe.  "host" pointers are caller-owned host memory (pageable or pinned); "dev" pointers
 * are caller-owned device memory.
 */
#ifndef XY_B200_H
#define XY_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct xy_state xy_state;   /* opaque */

enum { XY_INIT_COLD = 0,            /* all theta = +0.0f */
       XY_INIT_HOT  = 1 };          /* theta_i = (float)(2pi * (w0>>8) * 2^-24), w = Philox(seed; i, 0, INIT) */

enum { XY_OK = 0, XY_ERR_ARG = -1, XY_ERR_UNSUPPORTED_L = -2, XY_ERR_NOMEM = -3,
       XY_ERR_CUDA = -4, XY_ERR_STATE = -5 };

enum {
    XY_FLAG_LABELS64 = 1u,          /* hold labels as 64-bit words (default: 32-bit, enough for L <= 65536) */
    XY_FLAG_FOURIER = 2u            /* also reduce the structure-factor sums of every sweep (xy_fourier) */
};

enum { XY_OBS_NONE = 0,            /* chained sweeps do not reduce observables (thermalisation, throughput runs) */
       XY_OBS_ALL  = 1 };          /* every sweep reduces the sums of xy_obs (default) */

/* Observables of the configuration after `sweep` sweeps (PAPER.md:40 Eq. 3, :46-54 Eq. 4-6,
 * :107 Eq. 9).  All sums are un-normalised and accumulated in fp64.
 *   e_x = Cx/N, s_x = Sx/N,  Upsilon_x = <e_x> - beta N <s_x^2>,  <m^2> = <Mx^2+My^2>/N^2,  N = L^2. */
typedef struct {
    uint64_t sweep;                 /* T: number of sweeps done when this record was taken */
    double   beta;                  /* beta of sweep T-1 (NaN for T = 0 or after xy_set_sweep) */
    double   E, Mx, My;             /* E = -(Cx+Cy); Mx = sum cos theta_i; My = sum sin theta_i */
    double   Cx, Sx, Cy, Sy;        /* sum cos / sin (theta_i - theta_R(i)) and (theta_i - theta_D(i)) */
    uint64_t n_bonds_x, n_bonds_y, n_clusters;   /* of sweep T-1 (0 for T = 0) */
} xy_obs;

/* Structure-factor sums of one configuration at the smallest wave vector k = 2 pi / L, along x and
 * along y (Eq. 8-9: xi_2nd from chi(0) and chi(2 pi / L)):
 *   Fx = sum_r ( cos th cos kx, cos th sin kx, sin th cos kx, sin th sin kx ),  Fy: ky in place of kx;
 *   |sum_r s(r) e^{ikr}|^2 = Fx[0]^2 + Fx[1]^2 + Fx[2]^2 + Fx[3]^2.  Every term in fp64; agrees with
 *   the definition within 1e-9 N.  Recorded only by states created with XY_FLAG_FOURIER. */
typedef struct {
    uint64_t sweep;                 /* T: number of sweeps done when this record was taken */
    double   Fx[4], Fy[4];
} xy_fourier;

/* Schedule of the helicity-modulus PCC driver. */
typedef struct {
    uint64_t n_sweeps;              /* total sweeps of this call, including `discard` */
    uint64_t discard;               /* sweeps at beta0 before the first window (paper: 60000) */
    uint32_t window;                /* sweeps per beta*Upsilon estimate (paper: 1000); >= 1 */
    uint32_t dirs;                  /* 1: x links only (paper); 2: mean of x and y links */
    double   dbeta0;                /* informational copy of the initial step; the dbeta0 ARGUMENT wins */
    uint64_t halve_every;           /* halve dbeta every this many measured sweeps; 0 = never (paper) */
    double   dbeta_min;             /* floor for dbeta */
    double   target;                /* critical beta*Upsilon: 0.636508 or 2/pi */
} xy_pcc_schedule;

typedef struct {
    double   beta_final, dbeta_final;
    double   beta_mean;             /* mean of beta over the decisions of the last dbeta stage that has any */
    uint64_t n_decisions;
    double  *trace_beta;            /* optional caller-allocated host arrays (may be NULL): beta the window ran at */
    double  *trace_bY;              /*   and its beta*Upsilon estimate, one pair per decision */
    uint64_t trace_cap;             /* capacity of the two arrays (entries) */
    uint64_t trace_len;             /* out: number of decisions taken (may exceed trace_cap) */
} xy_pcc_out;

/* Controller state of the PCC driver: everything xy_pcc_continue needs beyond the configuration and the sweep counter
 * (checkpoint = xy_get_angles + xy_get_sweep + xy_pcc_get_state), and the sums of <m^2> and chi(2 pi / L) over the measured
 * sweeps fed to the controller so far, so that a long run needs no read-back of the per-sweep series. */
typedef struct {
    double   beta, dbeta;           /* beta of the next sweep, current step */
    double   acc_e, acc_s2;         /* sums of the open window */
    uint64_t k, n_decisions;        /* measured sweeps fed, decisions taken */
    double   stage_sum, last_sum;   /* beta_mean bookkeeping (O8) */
    uint64_t stage_cnt, last_cnt;
    double   sum_m2;                /* sum over the fed sweeps of (Mx^2 + My^2) / N^2 */
    double   sum_chik;              /* sum of (|F_x|^2 + |F_y|^2) / (2 N) (states with XY_FLAG_FOURIER, else 0) */
    uint64_t n_acc;                 /* number of sweeps in the two sums */
} xy_pcc_state;

/* ---- the five calls of the problem statement ------------------------------------------------ */

/* Create a state: L x L lattice, RNG seed, initial configuration XY_INIT_*; sweep counter t = 0.
 * Device memory is allocated with cudaMalloc and owned by the state.  L must be a multiple of 64
 * with 64 <= L <= 65536 (all sizes of PAPER.md:64), else XY_ERR_UNSUPPORTED_L. */
int xy_create(xy_state **out, uint32_t L, uint64_t seed, int init);

/* Run n Swendsen-Wang sweeps at inverse temperature beta (finite, >= 0).  Only ENQUEUES work on
 * cuda_stream (a cudaStream_t passed as void*; NULL = the legacy default stream) and returns;
 * the sweep counter advances by n.  xy_sw_sweeps(n) is identical to n calls of xy_sw_sweeps(1).
 * XY_ERR_STATE if the counter would reach 2^32 (the RNG takes 32 bits of it). */
int xy_sw_sweeps(xy_state *s, double beta, uint64_t n, void *cuda_stream);

/* Observables of the current configuration (after all enqueued sweeps).  Synchronises the
 * state's stream.  out: caller-owned host memory. */
int xy_measure(xy_state *s, xy_obs *out);

/* PCC run (raise beta by dbeta when beta*Upsilon < target, lower it otherwise), with
 * the whole control loop on the device; blocking.  Starts at the state's current configuration and
 * sweep counter, on the state's last-used stream.  Order of operations: DESIGN.md section 3 (O8). */
int xy_pcc_run(xy_state *s, double beta0, double dbeta0, const xy_pcc_schedule *sched, xy_pcc_out *out);

/* As xy_pcc_run, but the controller goes on from its state as it stands (after an earlier xy_pcc_run / xy_pcc_continue
 * of this state, or xy_pcc_set_state): a run of n1 + n2 sweeps equals xy_pcc_run(n1) followed by xy_pcc_continue(n2) with
 * discard = 0, bit for bit.  out->n_decisions and the trace count the decisions of THIS call. */
int xy_pcc_continue(xy_state *s, const xy_pcc_schedule *sched, xy_pcc_out *out);
int xy_pcc_get_state(xy_state *s, xy_pcc_state *out);
int xy_pcc_set_state(xy_state *s, const xy_pcc_state *in);

/* Free the state (and its device memory unless it was created on a caller workspace). */
int xy_destroy(xy_state *s);

/* ---- workspace-on-caller-memory variant (used by the PyTorch binding) ------------------------ */

/* Bytes of device workspace a state of size L with `flags` needs. */
int xy_workspace_bytes(uint32_t L, uint32_t flags, size_t *nbytes);

/* As xy_create, with XY_FLAG_* flags, optionally on caller-owned DEVICE memory dev_workspace of
 * nbytes >= xy_workspace_bytes (256-byte aligned; must outlive the state; xy_destroy then frees
 * only host resources).  dev_workspace == NULL: allocate internally. */
int xy_create_ex(xy_state **out, uint32_t L, uint64_t seed, int init, uint32_t flags,
                 void *dev_workspace, size_t nbytes);

/* ---- parity / checkpoint extensions (host buffers; each synchronises the state's stream) ----- */

/* the getters below copy the first n sites (row-major), 1 <= n <= L*L; the _range variants copy the n
 * sites first .. first+n-1 (first + n <= L*L), so any part of a lattice too large for host memory can be
 * inspected (label VALUES stay global site indices). */
int xy_get_angles(xy_state *s, float *host, size_t n);
int xy_get_angles_range(xy_state *s, float *host, uint64_t first, size_t n);
/* Replace the configuration (n = L*L values in [0, 6.2831855]).  The values are staged and range-checked
 * on the device BEFORE they replace theta: on XY_ERR_ARG the configuration is unchanged.  The labels of
 * the previous sweep are given up (their array is the staging area). */
int xy_set_angles(xy_state *s, const float *host, size_t n);
/* canonical labels of the most recent sweep, label = minimum site index of the cluster, widened
 * to int64 for every L; XY_ERR_STATE before the first sweep. */
int xy_get_labels(xy_state *s, int64_t *host, size_t n);
int xy_get_labels_range(xy_state *s, int64_t *host, uint64_t first, size_t n);
/* bonds of the most recent sweep, one byte per site: bit0 = x bond, bit1 = y bond. */
int xy_get_bonds(xy_state *s, uint8_t *host, size_t n);
int xy_get_bonds_range(xy_state *s, uint8_t *host, uint64_t first, size_t n);
/* Whole-lattice invariants of the most recent sweep's labels against its bonds, counted on the device
 * (for lattices whose label array does not fit host memory): counts[0] = #{label[i] > i},
 * counts[1] = #{label[label[i]] != label[i]}, counts[2] / counts[3] = active x / y bonds (periodic wrap
 * included) whose ends carry different labels, counts[4] = #{label[i] == i} (the number of clusters).
 * A correct labeling has counts[0..3] = 0 and counts[4] = xy_obs.n_clusters.  XY_ERR_STATE before the
 * first sweep. */
int xy_debug_check_labels(xy_state *s, uint64_t counts[5]);
/* per-sweep records for T = first_sweep .. first_sweep+count-1 from the device ring
 * (capacity xy_series_capacity(); records older than that are gone -> XY_ERR_ARG). */
int xy_get_series(xy_state *s, xy_obs *host, uint64_t first_sweep, uint64_t count);
int xy_series_capacity(xy_state *s, uint64_t *cap);
/* Structure-factor sums (states created with XY_FLAG_FOURIER; XY_ERR_STATE otherwise): of the current
 * configuration, and of the configurations after sweeps first_sweep .. first_sweep + count - 1 as far
 * as the device ring still holds them (same window as xy_get_series).  out / host: HOST memory. */
int xy_measure_fourier(xy_state *s, xy_fourier *out);
int xy_get_fourier_series(xy_state *s, xy_fourier *host, uint64_t first_sweep, uint64_t count);
/* Second-moment correlation length (Eq. 8) from chi(0) and chi(2 pi / L) of Eq. 9:
 *   *out = sqrt(chi0 / chik - 1) / (2 sin(pi / L)).
 * chi0 = <Mx^2 + My^2> / N and chik = <|Fx|^2 + |Fy|^2> / (2 N) are the caller's averages over measured sweeps (xy_obs and
 * xy_fourier records, or N * sum_m2 / n_acc and sum_chik / n_acc of xy_pcc_state).  Host arithmetic on two numbers; no
 * state, no GPU.  XY_ERR_ARG (and *out = NaN) unless L >= 2, chik > 0 and chi0 >= chik, all finite. */
int xy_xi2nd(double chi0, double chik, uint32_t L, double *out);
int xy_get_sweep(xy_state *s, uint64_t *t);
int xy_set_sweep(xy_state *s, uint64_t t);                      /* resume / sampled-sweep parity */
int xy_debug_fix_phi(xy_state *s, int on, double phi);          /* Ising-limit and 2x2-style tests */
/* XY_OBS_NONE: the following xy_sw_sweeps (and the `discard` sweeps of xy_pcc_run) skip the fp64
 * observable sums (the bond decisions, labels and angles are unchanged, bit for bit); their ring records
 * keep beta and the counts, the sums read NaN (so do the xy_fourier records of those sweeps, with their sweep
 * number set).  xy_measure still returns the sums of the current
 * configuration (one observables-only pass).  XY_OBS_ALL (default) restores the per-sweep series. */
int xy_set_obs_mode(xy_state *s, int mode);
/* number of bond decisions of all sweeps so far that the fp32 filter could not settle and that
 * were re-evaluated with the full fp64 expression. */
int xy_get_fallback_count(xy_state *s, uint64_t *count);

/* ---- measurement hooks (bench.py) ----------------------------------------------------------- */

/* on != 0: record CUDA events on the state's stream around every kernel of every following sweep
 * (k_bonds, k_label, k_merge, k_flip), so that per-kernel device time can be read back; off: stop. */
int xy_debug_kernel_timing(xy_state *s, int on);
/* Synchronise and return, accumulated since timing was switched on: device milliseconds and launch
 * counts of [0] k_bonds, [1] k_label, [2] k_merge, [3] k_flip.  Resets the accumulators. */
int xy_get_kernel_times(xy_state *s, double ms[4], uint64_t launches[4]);
/* Total number of kernels this state has launched so far (all kinds). */
int xy_get_launch_count(xy_state *s, uint64_t *count);

/* ---- step-level entry points for the parity tests -------------------------------------------- */

/* Run only the labeling kernels (tile-local union-find, boundary merge) on an injected bond set
 * (canonical byte layout as xy_get_bonds); read the result with xy_get_labels. */
int xy_label_bonds(xy_state *s, const uint8_t *host_bonds, size_t n);
/* Evaluate the CUDA path's own Philox4x32-10 device function on n (counter, key) pairs:
 * ctr_host[4n], key_host[2n] -> out_host[4n]. */
int xy_debug_philox(const uint32_t *ctr_host, const uint32_t *key_host, uint32_t *out_host, size_t n);
/* Same inputs through NVIDIA cuRAND's curand_Philox4x32_10 device function (independent pin). */
int xy_debug_curand_philox(const uint32_t *ctr_host, const uint32_t *key_host, uint32_t *out_host, size_t n);

/* Range-check counters of a library built with -DXY_CHECKED (every data-derived index of the kernels is
 * checked and violations counted: [0] sincos table entry, [1] tile-local parent offset, [2] wave-list site,
 * [3] label chased in global memory, [4] k_flip queue slot, [5] coin-table index).  *checked_build = 0 and
 * all zeros from the normal build, which compiles the checks away. */
int xy_debug_check_counts(uint64_t counts[8], int *checked_build);

/* ---- observables without any allocation ------------------------------------------------------
 * The sums E, Mx, My, Cx, Sx, Cy, Sy of xy_obs (PAPER.md:40 Eq. 3, :46-54 Eq. 4-6) of a configuration the CALLER holds
 * in device memory, for programs in which this library may not allocate device memory: a host application that has
 * handed the whole GPU to its own pool (a framework's caching allocator, a fixed per-job memory budget), so that a
 * cudaMalloc from a library can fail or fragment it; and loops that cannot afford the device-wide stall a cudaMalloc /
 * cudaFree implies while other streams are busy.  Every other way to these sums goes through a state, whose creation
 * allocates or needs a workspace of 8.4 bytes per site.
 *   dev_theta  in : L*L angles in DEVICE memory, row-major, each in [0, 6.2831855] as everywhere in this library
 *                   (not checked here: an angle outside that range makes the kernel fault); not modified.
 *   L             : a multiple of 64 with 64 <= L <= 65536; anything else is rejected with XY_ERR_UNSUPPORTED_L and
 *                   nothing is launched.
 *   dev_out    out: one xy_obs in DEVICE memory (8-byte aligned).  The seven sums are written; sweep, beta and the
 *                   three counts read 0.  The sums are the ones xy_measure returns for the same angles on the same
 *                   GPU (same kernel, same grid, same summation order).
 *   cuda_stream   : the work (two small memsets and one kernel) is only ENQUEUED there; NULL = legacy default stream.
 * Scratch: the per-CTA partial sums, the last-CTA ticket and the sine / cosine table sit in one file-scope device array
 * of 406 528 bytes (under 0.4 MiB) that every GPU which loads this library carries until the process ends.  All calls
 * on a device share it and find the previous call's contents in it; the call clears what has to start at zero.  Two
 * calls whose kernels can overlap on one GPU (different streams, or two host threads) therefore RACE: serialise them.
 * The first call on each device does the one-time set-up for that device (looks up the array's device address, uploads
 * the 103 KB table with a blocking copy, sets kernel attributes, synchronises the device), so make that first call
 * during start-up, on the device you will use, and before you begin any stream capture.
 * The call uses no cudaMalloc, cudaFree or allocating library routine, before or after set-up.
 * Errors: XY_ERR_ARG (NULL or non-device pointer), XY_ERR_UNSUPPORTED_L, XY_ERR_CUDA. */
int xy_observe_static(const float *dev_theta, uint32_t L, xy_obs *dev_out, void *cuda_stream);

/* ---- row-slab sharding across GPUs (SURVEY.md 8(e) / 8(f) #3; PAPER.md:34 "the inter-GPU labeling", :64) ----------
 * One state per rank holds rows [y_off, y_off + rows) of the L x L lattice (rows and y_off multiples of 32, fewer than
 * 2^31 sites -- L = 65536 therefore needs at least 4 slabs --, 32-bit labels) plus one halo row: the first row of the slab below (of rank 0 for the last rank).  Every
 * random number is keyed by the site's index in the WHOLE lattice, so G slabs reproduce the sweep of one L x L state
 * bit for bit.  One sweep at counter t is
 *     xy_slab_label   (every rank)  direction, bonds, local labels (tile labeling + merge inside the slab), edge record
 *     all-gather of the ranks' edge records (caller: NCCL / any transport), in rank order
 *     xy_slab_flip    (every rank)  replicated union-find over the cut roots, overrides, coins by canonical root, flip
 *     exchange of first rows -> halo rows (caller), before the next xy_slab_label or xy_measure.
 * xy_measure / xy_get_series return the slab's PARTIAL sums (its sites; the y links of its last row use the halo row;
 * n_clusters counts the clusters whose canonical root lies in the slab): the caller adds the ranks' records.
 * The halo row is valid from creation (cold: zeros; hot: the initial values of that row of the whole lattice).  Edge sites
 * of this rank's gathered record that lie outside the slab (wrong rank / nranks, records out of rank order) are skipped
 * by xy_slab_flip and reported as XY_ERR_ARG by the next xy_measure or xy_get_labels of the slab.
 * xy_get_labels returns canonical labels of the whole lattice (after xy_slab_flip).  xy_sw_sweeps, xy_pcc_run,
 * xy_label_bonds and xy_debug_check_labels return XY_ERR_STATE on a slab. */
int xy_slab_workspace_bytes(uint32_t L, uint32_t rows, uint32_t flags, size_t *nbytes);
int xy_slab_create(xy_state **out, uint32_t L, uint32_t rows, uint32_t y_off, uint64_t seed, int init, uint32_t flags,
                   void *dev_workspace, size_t nbytes);      /* dev_workspace NULL: the library allocates */
/* device pointers (inside the workspace) of the buffers the caller exchanges: the slab's first row (send), its halo
 * row (receive: row_bytes = 4 L), and its edge record (send: edge_bytes; layout: u64 root of every site of the first
 * row, u64 root of every site of the last row, as site indices of the whole lattice, then one byte per site of the
 * last row: its +y bond) */
int xy_slab_buffers(xy_state *s, void **dev_first_row, void **dev_halo_row, size_t *row_bytes, void **dev_edges, size_t *edge_bytes);
int xy_slab_label(xy_state *s, double beta, void *cuda_stream);
/* parity hook: the label phase on an injected bond set of the slab's sites (canonical bytes as xy_get_bonds); the
 * following xy_slab_flip stitches (and flips with the coins of the current sweep counter) */
int xy_slab_label_bonds(xy_state *s, const uint8_t *host_bonds, size_t n);
/* dev_gathered_edges: nranks edge records in rank order (device memory).  The table of the replicated union-find is part
 * of the workspace, sized for L / rows slabs; only a call with another nranks allocates (once) a table of its own. */
int xy_slab_flip(xy_state *s, const void *dev_gathered_edges, uint32_t nranks, uint32_t rank, void *cuda_stream);
/* The PCC driver on a sharded lattice (the paper's own use of its multi-GPU code, PAPER.md:62-66 at L >= 8192): the
 * controller (O8) runs replicated on every rank's device, fed with all-reduced sums.  Per measured sweep, after the halo
 * exchange: xy_slab_obs_partial (the slab's six sums of the new configuration -> dev_partial8), all-reduce (sum) of the 8
 * doubles into dev_global8 (caller), xy_slab_pcc_feed.  xy_slab_label_pcc sweeps at the controller's beta.  The
 * controller state is read with xy_pcc_get_state; all ranks hold the same one. */
int xy_slab_pcc_setup(xy_state *s, double beta0, double dbeta0, const xy_pcc_schedule *sched);
int xy_slab_label_pcc(xy_state *s, void *cuda_stream);
int xy_slab_pcc_buffers(xy_state *s, void **dev_partial8, void **dev_global8);
int xy_slab_obs_partial(xy_state *s, void *cuda_stream);
int xy_slab_pcc_feed(xy_state *s, void *cuda_stream);

/* ---- q-state Potts model on the same labeling core ------------------------
 * PAPER.md:30-34 cites the authors' GPU Swendsen-Wang codes for the Potts and Ising models (refs 19, 22)
 * as the origin of the labeling method; the update rule is not restated there and is the textbook one
 * (readings P1-P5).  H = -J sum_<ij> delta(s_i, s_j), J = 1, s_i in {0..q-1} held as
 * one byte per site, L x L periodic, same site and bond indexing as above.  One sweep at counter t:
 *   bonds  <ij> active iff s_i == s_j and u < 1 - exp(-beta), u the site's bond uniform of the XY sweep;
 *   labels as above (k_label / k_merge unchanged);
 *   spins  every cluster takes s = floor(q w / 2^32), w = word (rho & 3) of Philox(seed; rho >> 2, t, POTTS),
 *          rho the cluster's label.
 * q = 2 is the Ising model at coupling beta / 2.  Labels are 32-bit.  Same error codes as above. */
typedef struct xy_potts xy_potts;   /* opaque */

typedef struct {
    uint64_t sweep;                 /* T: sweeps done */
    double   beta;                  /* beta of sweep T-1 (NaN before the first sweep) */
    int64_t  E;                     /* -(ex + ey) */
    uint64_t ex, ey;                /* x / y links with equal spins in the current configuration */
    uint64_t count[16];             /* sites per spin value (entries >= q are 0) */
    uint64_t n_bonds_x, n_bonds_y, n_clusters;   /* of sweep T-1 (0 before the first sweep) */
} xy_potts_obs;

/* L as for xy_create; 2 <= q <= 16; init XY_INIT_COLD (all 0) or XY_INIT_HOT (s_i = floor(q w0 / 2^32) of the
 * INIT call of site i).  The library allocates the device workspace (about 5.4 bytes per site + 16 MiB). */
int xy_potts_create(xy_potts **out, uint32_t L, uint32_t q, uint64_t seed, int init);
int xy_potts_destroy(xy_potts *s);
/* n sweeps at beta (finite, >= 0), enqueued on cuda_stream (cudaStream_t, NULL = default); does not block. */
int xy_potts_sweeps(xy_potts *s, double beta, uint64_t n, void *cuda_stream);
/* observables of the current configuration (one counting pass); blocks until the stream is idle */
int xy_potts_measure(xy_potts *s, xy_potts_obs *out);
/* host buffers: the first n spins (n <= L*L); all L*L spins, rejected with XY_ERR_ARG (state unchanged) if any is >= q */
int xy_potts_get_spins(xy_potts *s, uint8_t *host, size_t n);
int xy_potts_set_spins(xy_potts *s, const uint8_t *host, size_t n);
int xy_potts_get_sweep(xy_potts *s, uint64_t *t);
int xy_potts_set_sweep(xy_potts *s, uint64_t t);
/* bonds (byte per site: bit0 = +x, bit1 = +y) and canonical labels (minimum site index) of the last sweep */
int xy_potts_get_bonds(xy_potts *s, uint8_t *host, size_t n);
int xy_potts_get_labels(xy_potts *s, int64_t *host, size_t n);
int xy_potts_get_launch_count(xy_potts *s, uint64_t *count);

const char *xy_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* XY_B200_H */

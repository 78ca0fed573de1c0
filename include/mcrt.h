/*
 * mcrt.h -- C ABI of the B200-native photon-packet transport library (libmcrt_b200.so).
 *
 * The library implements the hot path of the 3-D Monte Carlo dust radiative-transfer method of
 * Heymann & Siebenmorgen (arxiv 1203.2941; citations are lines of /root/reference/PAPER.md):
 * packets emitted by a point source walk cell by cell through a Cartesian dust grid (PAPER.md:45-53,
 * Eq. 2-3), scatter with Henyey-Greenstein sampling (Eq. 15 at PAPER.md:203) or are
 * absorbed and immediately re-emitted Bjorkman & Wood style (Eq. 4, 5, 10),
 * while absorption counts, Lucy path-length tallies (Eq. 9) and the escape SED
 * are accumulated.  Every step runs in hand-written CUDA kernels for sm_100a.
 *
 * Conventions
 *  - Every call returns an int: MCRT_OK (0) or a negative MCRT_E* code.  No exception or abort crosses
 *    the ABI; mcrt_last_error() returns the message of the last failure of that context.
 *  - Pointers are HOST pointers unless the call takes an `mcrt_mem where` argument, in which case the
 *    array arguments marked [where] live in host memory (MCRT_HOST) or in device memory of the
 *    context's device (MCRT_DEVICE).  The caller owns every array it passes and may free or reuse it
 *    as soon as the call returns (the library copies what it keeps).  Outputs go to caller-allocated
 *    buffers; a NULL output pointer skips that output.
 *  - Grid arrays are [nz][ny][nx] with x the fastest index; the grid spans [0,nx*h]x[0,ny*h]x[0,nz*h].
 *  - Frequency tables are [n_species][n_nu] on an ascending frequency grid.
 *  - All work is issued on the context's stream (default: the legacy default stream; see
 *    mcrt_set_stream).  Calls that return data to the host synchronise that stream.
 *  - One context = one device (the current device at mcrt_grid_create) = one stream.  A context is
 *    not thread safe.
 *  - Call order: mcrt_grid_create -> mcrt_dust_tables -> mcrt_source -> [mcrt_escape_bins] ->
 *    mcrt_run (any number of times) -> mcrt_read / mcrt_read_raw -> mcrt_destroy.  Out-of-order calls
 *    return MCRT_ESTATE.
 */
#ifndef MCRT_H_
#define MCRT_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct mcrt_ctx mcrt_ctx; /* opaque */

typedef enum { MCRT_HOST = 0, MCRT_DEVICE = 1 } mcrt_mem;

enum {
    MCRT_OK = 0,
    MCRT_EINVAL = -1,   /* bad argument (message says which) */
    MCRT_ESTATE = -2,   /* call out of order */
    MCRT_ENOMEM = -3,   /* workspace too small / allocation failed */
    MCRT_ECUDA = -4,    /* CUDA runtime error */
    MCRT_EOVERFLOW = -5 /* a fixed-point Lucy tally exceeded 2^62 (also returned by the read calls: the tallies
                           they would hand back have wrapped) */
};

typedef enum {
    MCRT_MODE_BW_EPOCH = 0,      /* Bjorkman & Wood immediate re-emission, Eq. 10, deterministic epochs */
    MCRT_MODE_FROZEN_T_SWEEP = 1,/* iterative scheme of PAPER.md:73: T frozen per sweep, Eq. 5 */
    MCRT_MODE_LIVE_BW = 2        /* Bjorkman & Wood as printed: the temperature follows every single
                                    absorption (atomic count with return, Eq. 4 inverted on the spot), all packets in one
                                    launch.  The count a packet sees depends on the order of the atomics: results are
                                    reproducible only statistically.  For comparison with the epochs. */
} mcrt_mode;

/* Options of mcrt_run.  Fill with mcrt_default_opts() first. */
typedef struct {
    int32_t mode;              /* mcrt_mode */
    uint64_t epoch_B0;         /* first epoch size; 0 = max(256, largest power of two <= N/256) */
    uint64_t epoch_Bmax;       /* largest epoch size; 0 = 2^22.  Epoch e has min(B0*2^e, Bmax) packets */
    int32_t n_sweeps;          /* MCRT_MODE_FROZEN_T_SWEEP: number of sweeps (each emits N packets) */
    int32_t sweep_T_from_lucy; /* sweeps take T from the Lucy tally (1) or from absorption counts (0) */
    int32_t record_digests;    /* keep a per-packet event digest (needs digest capacity in the workspace) */
    int32_t reset_tallies;     /* zero all tallies before the run (default 1) */
    uint32_t rng_pass;         /* 4th Philox counter word of the B&W run; sweep s uses rng_pass + s */
    int32_t grid_blocks;       /* launch tuning, 0 = auto.  Results never depend on it. */
    int32_t block_threads;     /* launch tuning, 0 = auto (multiple of 32, <= 512) */
    int32_t time_kernels;      /* bracket every kernel with CUDA events on the context's stream; the
                                  summed durations are returned in mcrt_run_stats (transport_ms, update_ms) */
    uint64_t first_packet_id;  /* the run's packets have ids first_packet_id .. first_packet_id + n_packets - 1
                                  (a packet's random stream is keyed by its id, north_star item 1) */
    uint64_t n_total;          /* the luminosity is split into this many packets, xi = L / n_total;
                                  0 = n_packets.  Lets several runs (reset_tallies = 0, disjoint id ranges) add up
                                  to one run of n_total packets */
    double epoch_growth;       /* epoch e+1 has min(floor(B_e * growth), Bmax) packets; 0 = 2.0; must be >= 1 */
    int32_t part_index;        /* partitioned run (packets are independent): this context transports */
    int32_t part_count;        /* slice part_index of part_count of EVERY epoch's id range; 0 or 1 = the whole run */
    uint32_t source_strata;    /* > 0: stratified source frequencies (Eq. 1: equal-energy source bins with
                                  equally many packets): packet id takes stratum id mod source_strata of the cumulative
                                  source spectrum and a uniform position in it.  0 (default): plain sampling */
    uint32_t carry_interactions; /* MCRT_MODE_BW_EPOCH: > 0 = a packet that has had this many interactions within one
                                  epoch stops behind the last of them and continues in the next epoch, from the same
                                  state and random stream, at that epoch's temperatures; packets still carried after
                                  the last epoch run in further epochs, the budget doubling each time.  The
                                  deterministic restatement of the pause / resume of PAPER.md:128-130 (paper: 100).
                                  0 (default) = no limit.  <= 65535; not in partitioned runs.  The list of carried
                                  packets is allocated with cudaMalloc (88 bytes per packet of an epoch). */
    int32_t no_hot_cells;      /* launch tuning: 1 = do not keep per-CTA copies of the tallies of the cells around the
                                  source (default 0: kept; the sums are integers, so results do not depend on it) */
    int32_t lucy_hybrid;       /* 1 = the thresholded estimator of Sect. 3.1 (readings Q37-Q39): only cells whose
                                  maximal optical depth sqrt(3) h rho max_nu(kabs+ksca) is below 10^-2 are tallied, with Eq. 9's
                                  (1 - e^-tau_abs) per traversal, and their temperature (per-epoch index, sweeps, the T_lucy of
                                  mcrt_read) comes from that energy; all other cells' from their counts.  Default 0: the linear
                                  path-length tally in every cell.  Not with mixtures, live B&W or partitioned runs; a run that
                                  continues stored tallies (reset_tallies = 0, sweeps) must use the estimator that made them */
    int32_t tau_redraw_per_cell; /* 1 = the optical depth to the next interaction is drawn anew on entering every cell, the paper's
                                  literal form (footnote 1, states its equivalence with one draw per
                                  flight, which pin P11 confirms statistically): the cell reached after c crossings of a flight
                                  uses Philox draw (flight's draw index + c).  Default 0: one draw per flight (reading Q4).
                                  Trajectories differ from the default's; not with carry-over or live B&W */
} mcrt_run_opts;

/* Counters of the runs since the last reset (all exact integers). */
typedef struct {
    uint64_t packets;          /* packets emitted */
    uint64_t crossings;        /* cell faces crossed, including the final exit */
    uint64_t dusty_crossings;  /* of those, traversed cells with rho > 0 */
    uint64_t flights;          /* optical-depth draws: packets + scatterings + absorptions */
    uint64_t scatterings;
    uint64_t absorptions;
    uint64_t escapes;
    uint64_t direct_escapes;   /* escaped without any interaction */
    uint64_t epochs;           /* transport-kernel launches */
    uint64_t lucy_adds;        /* fixed-point tally additions */
    uint64_t gpu_launches;     /* all kernels launched by mcrt_run */
    int32_t fx_bits;           /* fraction bits of the Lucy fixed point, min(40, 58 - ceil(log2 N)) */
    int32_t overflow;          /* 1 if some |tally| exceeded 2^62 */
    double transport_ms;       /* summed device time of the transport kernel launches (time_kernels = 1) */
    double update_ms;          /* summed device time of the per-epoch update / range-check kernels */
} mcrt_run_stats;

/* Per-packet digest used by the parity tests: 64-bit FNV-1a style hash over the packet's events
 * (EMIT, SCATTER, ABSORB, ESCAPE; each with cell index and frequency bin) and its counts. */
typedef struct {
    uint64_t hash;
    uint32_t crossings, scatterings, absorptions, escape_bin;
} mcrt_digest;

/* Bytes of device workspace a context of these sizes needs (pure function).  n_digests = capacity of
 * the per-packet digest buffer (0 if digests are never recorded). */
int mcrt_workspace_bytes(int nx, int ny, int nz, int n_species, int n_nu, int n_T, int n_dir,
                         uint64_t n_digests, size_t *bytes_out);

/* Create a context for an nx*ny*nz grid of cubic cells of edge cell_size_cm.
 *  rho      [where] float  [nz][ny][nx], dust mass density in g cm^-3, finite and >= 0 (0 = vacuum)
 *  species  [where] uint8  [nz][ny][nx], dust species of the cell, < n_species (1 <= n_species <= 255)
 *  workspace  device pointer to workspace_bytes bytes owned by the caller (e.g. a torch tensor) that
 *             must stay valid until mcrt_destroy, or NULL to let the library cudaMalloc its memory.
 *             256-byte alignment required.  The library sub-allocates from it in call order (grid
 *             here, tables in mcrt_dust_tables, histograms and digests at the first mcrt_run that
 *             needs them) and returns MCRT_ENOMEM when it runs out; size it with mcrt_workspace_bytes.
 *  nx, ny <= 2040, nz <= 1016 and at most 2^30 cells with the guard shell (cell coordinates are carried packed in 32 bits).
 * The grid is re-laid out on the device into bricks of packed 8-byte cell words (4x4x4 cells up to 256^3,
 * 8x8x8 up to 512^3, ...); a bit mask of the bricks without dust and, for each of them, a large box of empty
 * bricks around it are built here as well (they let packets cross vacuum without touching memory). */
int mcrt_grid_create(mcrt_ctx **out, int nx, int ny, int nz, double cell_size_cm, const float *rho,
                     const uint8_t *species, int n_species, mcrt_mem where, void *workspace,
                     size_t workspace_bytes);

/* Dust cross sections per species on the frequency grid and the temperature
 * grid of the T(E) and re-emission tables (Eq. 4, 5, 10).  Host pointers.
 *  nu_hz [n_nu] strictly ascending; kappa_abs, kappa_sca [n_species][n_nu] in cm^2 g^-1, >= 0 with
 *  kappa_abs + kappa_sca > 0; g [n_species][n_nu] with |g| < 1; T_grid [n_T] strictly ascending, K.
 *  2 <= n_nu <= 65535, 2 <= n_T <= 65535.  May be called once per context. */
int mcrt_dust_tables(mcrt_ctx *ctx, int n_nu, const double *nu_hz, const double *kappa_abs,
                     const double *kappa_sca, const double *g, int n_T, const double *T_grid);

/* Dust mixtures with per-material temperatures ("two populations of large grains",
 * PAPER.md:43 "different grain materials", "the total number of absorbed photon packets per particle and
 * cell is used to calculate the temperature of each material").  After mcrt_dust_tables, before the first run, once
 * per context: redefines cell species x (the byte of the grid's species array, x < n_species) as a MIXTURE of
 * n_components[x] = 1 or 2 of the n_species materials of mcrt_dust_tables: component c of x is material
 * material[2x+c] with mass fraction fraction[2x+c] > 0 of the cell's density (the fractions of x add up to 1).
 * Host pointers, [n_species], [n_species][2], [n_species][2].  The paper has no formulas for this; the readings
 * (Q34-Q36): extinction adds up, kext_x = (f0 kabs0 + f0 ksca0) + (f1 kabs1 + f1 ksca1); the ONE uniform
 * number z that decides scattering against absorption also picks the component, in proportion to its
 * share of kext_x -- z < f0 ksca0/kext_x: scattered by component 0 (its g), z < albedo_x: by component 1,
 * z < albedo_x + f0 kabs0/kext_x: absorbed by component 0, else by component 1; every component keeps its own
 * absorption count, Lucy tally (f_c kabs_c rho ds per traversal) and temperature (Eq. 4 with its material and its
 * mass rho f_c V), and re-emits what it absorbed from its own Eq. 10 / Eq. 5 row.  mcrt_read / mcrt_read_raw return
 * component 0, mcrt_read_component either.  A one-component mixture is that material, bit for bit.
 * Not available with MCRT_MODE_LIVE_BW, in partitioned runs and for mcrt_ray_trace (MCRT_EINVAL); such runs use
 * the kernel instantiation of the rarely used features and no per-CTA hot-cell copies. */
int mcrt_dust_mixtures(mcrt_ctx *ctx, const int32_t *n_components, const int32_t *material, const double *fraction);

/* One level of refinement ("Each cube is divided into an arbitrary number of sub-cubes
 * of volume V_i and constant density rho_i ... a finer sampling whenever required").  Reading Q40: the n_sub
 * cubes with the cell indices cube[n_sub] ((iz ny + iy) nx + ix; each at most once; their own density in the grid must
 * be > 0, a placeholder) are divided into R x R x R equal sub-cubes, R = 2, 4 or 8, with the densities rho_sub
 * [n_sub][R^3] (g cm^-3, >= 0; order z, y, x) and species species_sub [n_sub][R^3].  Packets cross them with the same
 * cell walk on the lattice of sub-cube faces; every sub-cube is a cell of its own for optical depth, Lucy tally,
 * absorption count and temperature (Eq. 4 with V = (h/R)^3); in digests its cell number is nx ny nz + b R^3 +
 * (gz R + gy) R + gx for sub-cube (gx, gy, gz) of cube cube[b].  With every cube divided the run is the run on the
 * (n R)^3 uniform grid, bit for bit.  Host pointers.  After mcrt_grid_create, before the first run, once per context
 * (after a failure the context must be destroyed).  mcrt_read / mcrt_read_raw return 0 for a divided cube itself;
 * mcrt_read_subcells returns the sub-cubes' outputs.  Not with mixtures, carry-over, the thresholded estimator, live
 * B&W, partitioned runs or mcrt_ray_trace; such runs use the kernel instantiation of the rarely used features. */
int mcrt_subgrid(mcrt_ctx *ctx, int R, uint64_t n_sub, const int64_t *cube, const float *rho_sub,
                 const uint8_t *species_sub);

/* The arrays of mcrt_read and mcrt_read_raw for the sub-cubes, [n_sub R^3] each in the order of mcrt_subgrid; any
 * pointer may be NULL. */
int mcrt_read_subcells(mcrt_ctx *ctx, double *E_abs_count, double *E_abs_lucy, float *T_count, float *T_lucy,
                       uint64_t *k_abs, int64_t *lucy_fx, uint16_t *tidx, mcrt_mem where);

/* Point source: luminosity L_erg_s split into equal-energy packets xi = L/N.
 *  T_star_K > 0: blackbody spectrum; otherwise L_nu_weights [n_nu] gives the spectral shape L_nu at the
 *  grid frequencies (any normalisation, >= 0, not all zero).  pos_cm strictly inside the grid. */
int mcrt_source(mcrt_ctx *ctx, double L_erg_s, double T_star_K, const double *L_nu_weights,
                const double pos_cm[3]);

/* Escape histogram bins in |cos i|: abs_mu_edges [n_dir+1] ascending from 0 to 1.
 * Default (if never called): one bin. */
int mcrt_escape_bins(mcrt_ctx *ctx, int n_dir, const double *abs_mu_edges);

void mcrt_default_opts(mcrt_run_opts *opts);

/* Transport n_packets packets with ids opts.first_packet_id .. + n_packets - 1 ("follow all N
 * photon packets ... until they ... escape").  opts NULL = defaults.  If stats_out is NULL the call only
 * enqueues work on the stream and returns without synchronising (a fixed-point overflow is then reported by the
 * next mcrt_get_stats / mcrt_read / mcrt_read_raw as MCRT_EOVERFLOW); otherwise it synchronises and fills
 * stats_out.  With reset_tallies = 0 the run adds to the stored tallies; that is refused (MCRT_ESTATE) when their
 * packet energy xi or fixed-point scale differs from this run's (use n_total). */
int mcrt_run(mcrt_ctx *ctx, uint64_t n_packets, uint64_t seed, const mcrt_run_opts *opts,
             mcrt_run_stats *stats_out);

/* The same run one step at a time: mcrt_run(...) == mcrt_run_begin; while (!done) mcrt_run_step; mcrt_run_end.
 * A step is one epoch (per-cell temperature-index update + transport of that epoch's packets) in
 * MCRT_MODE_BW_EPOCH and one whole sweep in MCRT_MODE_FROZEN_T_SWEEP.  Only enqueues work on the stream.
 * In a PARTITIONED run (opts.part_count > 1) every part calls the same sequence with the same
 * n_packets / seed / opts except part_index, and after EVERY step the parts' tallies must be summed:
 *   mcrt_exchange_begin (each part) -> element-wise 64-bit integer sum over the parts of every listed array,
 *   written back to every part (ncclAllReduce(ncclSum, ncclInt64) in place, or mcrt_exchange_peer_sum) ->
 *   mcrt_exchange_end (each part).
 * The next mcrt_run_step / mcrt_run_end of a partitioned run returns MCRT_ESTATE until that has happened.  All
 * tallies are integers, so the result is bit-identical to the unpartitioned run. */
int mcrt_run_begin(mcrt_ctx *ctx, uint64_t n_packets, uint64_t seed, const mcrt_run_opts *opts);
int mcrt_run_step(mcrt_ctx *ctx, int *done_out);
int mcrt_run_end(mcrt_ctx *ctx, mcrt_run_stats *stats_out /* NULL: do not synchronise */);

/* Arrays of 64-bit integers (DEVICE pointers into the context's memory) to be summed over the parts now. */
typedef struct {
    int32_t n;            /* number of arrays (<= 8) */
    void *ptr[8];
    uint64_t words[8];    /* length of each array in 64-bit words (the same on every part) */
} mcrt_exchange;

/* After a step of a partitioned run.  Between two epochs of a B&W run only the absorption counts are listed
 * (as this epoch's own increments; the temperature update is all that needs them); after the last epoch, and
 * after every sweep, also the Lucy tallies, both escape histograms and the run counters. */
int mcrt_exchange_begin(mcrt_ctx *ctx, mcrt_exchange *out);
int mcrt_exchange_end(mcrt_ctx *ctx);

/* The sum itself over peer-visible device memory (parts on one device, or on NVLink peers whose memory has been
 * mapped into this process with CUDA IPC / peer access): views[p] is part p's mcrt_exchange.
 *  phase 0 (reduce-scatter): this part sums slice part_index of every array over all parts into its own copy;
 *  phase 1 (all-gather): this part copies every other slice from the part that owns it.
 * All parts must have finished phase 0 before any starts phase 1 (stream order on one device, a barrier across
 * processes).  Runs on ctx's stream; n_parts <= 16. */
int mcrt_exchange_peer_sum(mcrt_ctx *ctx, int part_index, int n_parts, const mcrt_exchange *views, int phase);

/* Convenience for parts that live in ONE process on ONE device (tests): begin + both phases + end for all. */
int mcrt_exchange_local(mcrt_ctx *const *parts, int n_parts);

/* Pure host helpers (no device needed), so that every part of a partitioned run derives the same schedule:
 * mcrt_epoch_schedule writes the epoch sizes of a B&W run of n_packets (B0 / Bmax / growth as in mcrt_run_opts, 0 =
 * default) to sizes_out[0 .. min(n, max_epochs) - 1] and the epoch count n to *n_epochs_out; mcrt_part_slice gives
 * the slice [lo, hi) of an id range of `count` packets that part part_index of part_count transports
 * (lo = floor(count * r / R), hi = floor(count * (r + 1) / R): the slices tile the range). */
int mcrt_epoch_schedule(uint64_t n_packets, uint64_t epoch_B0, uint64_t epoch_Bmax, double epoch_growth,
                        uint64_t *sizes_out, uint64_t max_epochs, uint64_t *n_epochs_out);
int mcrt_part_slice(uint64_t count, int part_index, int part_count, uint64_t *lo_out, uint64_t *hi_out);

/* Measurement aid (configurations whose arrays fit L2 are reported against a MEASURED L2 read
 * bandwidth): `repeats` timed launches (after two warm-up launches), each sweeping a device buffer of `bytes`
 * bytes with 16-byte loads from every SM until about 4 GB have been read; returns the best read rate in GB/s.
 * A buffer far below the L2 size measures L2, a far larger one HBM. */
int mcrt_measure_read_bandwidth(size_t bytes, int repeats, double *gb_per_s_out);

/* Synchronise and return the counters accumulated since the last reset. */
int mcrt_get_stats(mcrt_ctx *ctx, mcrt_run_stats *stats_out);

/* Physical outputs, [where] arrays of the grid shape [nz][ny][nx] unless noted:
 *  E_abs_count  double, k * xi: absorbed luminosity per cell from absorption counts, erg s^-1 (Eq. 4)
 *  E_abs_lucy   double, path-length estimate of the same quantity (Eq. 9, linear form)
 *  T_count, T_lucy  float, dust temperature from either estimate by inverting Eq. 4 (0 where rho = 0
 *               or nothing was absorbed; clamped to the T grid)
 *  SED          double [n_dir][n_nu], escaping L_nu per solid angle, erg s^-1 Hz^-1 sr^-1 */
int mcrt_read(mcrt_ctx *ctx, double *E_abs_count, double *E_abs_lucy, float *T_count, float *T_lucy,
              double *SED, mcrt_mem where);

/* Raw integer tallies (parity tests), [where]: k_abs uint64 [cells]; lucy_fx int64 [cells];
 * sed_counts, sed_direct uint64 [n_dir][n_nu]; tidx uint16 [cells] (temperature index of the last
 * epoch); digests [n_packets of the last run] (only if recorded). */
/* Outputs of one component of the mixtures (mcrt_dust_mixtures; component 0 or 1): the arrays of mcrt_read and the
 * raw tallies of mcrt_read_raw for that component, [cells] each, any pointer may be NULL.  T is 0 where the cell's
 * mixture has no such component.  MCRT_ESTATE without mixtures. */
int mcrt_read_component(mcrt_ctx *ctx, int component, double *E_abs_count, double *E_abs_lucy, float *T_count,
                        float *T_lucy, uint64_t *k_abs, int64_t *lucy_fx, uint16_t *tidx, mcrt_mem where);

int mcrt_read_raw(mcrt_ctx *ctx, uint64_t *k_abs, int64_t *lucy_fx, uint64_t *sed_counts,
                  uint64_t *sed_direct, uint16_t *tidx, mcrt_digest *digests, mcrt_mem where);

/* ---- Scattering-event store and ray tracer (Sect. 4, Eq. 11-17) ----
 * "The index of the cell, the frequency of the scattered photon and the incoming direction is stored":
 * after mcrt_scatter_store every run appends one record per scattering at one of the listed frequency bins
 * (n_bins <= 16 indices into the frequency grid) to a list of `capacity` records in device memory (cudaMalloc; 12
 * bytes each).  A B&W run with reset_tallies and every frozen-T sweep start an empty list.  Events beyond the
 * capacity are counted, not kept.  The order of the records depends on scheduling; the multiset does not. */
typedef struct {
    uint32_t cell;      /* [nz][ny][nx] index */
    uint16_t slot;      /* position of the event's frequency bin in nu_bins */
    int16_t q[3];       /* incoming direction, q_a = rint(32767 u_a) */
} mcrt_scatter_event;
int mcrt_scatter_store(mcrt_ctx *ctx, int n_bins, const int32_t *nu_bins, uint64_t capacity);
/* *n_total_out = events counted; events [where], if not NULL, receives the first min(counted, capacity, max_events). */
int mcrt_scatter_events(mcrt_ctx *ctx, uint64_t *n_total_out, mcrt_scatter_event *events, uint64_t max_events,
                        mcrt_mem where);

/* The image of Sect. 4 at frequency bin nu_bin for an observer at distance_cm in direction e_z (from the object
 * towards the observer; need not be normalised), parallel projection (Eq. 11): pixel (a, b) of nx x ny square pixels
 * of pixel_cm looks along r = i0 + (a + 1/2 - nx/2) pixel e_x + (b + 1/2 - ny/2) pixel e_y + s e_z, i0 the centre of
 * the grid, e_x made orthogonal to e_z, e_y = e_z x e_x.  From the observer's side inwards every cell adds (Eq. 12, 17)
 *     A_pix / D^2 (I_e + I_s) exp(-tau),  tau = absorption optical depth between the cell and the observer (Eq. 13),
 *     I_e = (1 - exp(-tau_cell)) B_nu(T)  (Eq. 14; T from the counts, or from the Lucy tally if T_from_lucy),
 *     I_s = l / V sum over the cell's stored events of P_HG(beta) xi / dnu  (Eq. 15, 16; beta between e_z and the
 *           event's incoming direction; l = path length in the cell, V its volume).
 * F_emission, F_scatter: [where] double [ny][nx], erg s^-1 cm^-2 Hz^-1 (F_scatter may be NULL; it is zero unless
 * nu_bin is being stored).  Needs a finished run. */
typedef struct {
    double e_z[3], e_x[3];
    int32_t nx, ny;
    double pixel_cm, distance_cm;
    int32_t nu_bin, T_from_lucy;
} mcrt_image_opts;
int mcrt_ray_trace(mcrt_ctx *ctx, const mcrt_image_opts *opts, double *F_emission, double *F_scatter, mcrt_mem where);

/* Host copies of the derived tables (tests): dnu [n_nu], J [n_species][n_T], cdf_B and cdf_dB
 * [n_species][n_T][n_nu], albedo [n_species][n_nu], src_cdf [n_nu]. */
int mcrt_read_tables(mcrt_ctx *ctx, double *dnu, double *J, double *cdf_B, double *cdf_dB, double *albedo,
                     double *src_cdf);

/* Raw Philox-4x32-10 blocks computed ON THE DEVICE for n (counter, key) pairs given on the host
 * (ctr [n][4], key [n][2], out [n][4]); lets the tests pin the device generator. */
int mcrt_philox_device(const uint32_t *ctr, const uint32_t *key, uint32_t *out, uint64_t n);

/* The trajectory's elementary functions computed ON THE DEVICE for n host values z in (0,1): ln z (used as
 * tau = -ln zeta) and sin / cos of 2 pi z (azimuth).  They are explicit fp64
 * algorithms (reading Q28), so the tests can demand bit-equality with the oracle's. */
int mcrt_traj_math_device(const double *z, double *ln_z, double *sin_2piz, double *cos_2piz, uint64_t n);

/* The same functions through an entry point that ALLOCATES NOTHING (no cudaMalloc / cudaFree, no host allocation), for
 * callers that cannot allocate: tight loops, harnesses that forbid it.  Host pointers as above; n <= MCRT_STATIC_MAX_N,
 * beyond that MCRT_EINVAL with a message.  The device copies of z and of the three results live in a static device
 * array of 4 x MCRT_STATIC_MAX_N doubles (2 MiB) that every GPU which loads the library holds until the process exits
 * and that ALL calls share: it keeps the last call's contents (nothing in it has to start at zero -- a call reads back
 * only what it wrote), and calls that overlap on the GPU (several host threads) race on it -- serialise them.  Runs on
 * the current device, default stream, synchronous.  Results are bit-identical to mcrt_traj_math_device. */
#define MCRT_STATIC_MAX_N 65536
int mcrt_traj_math_device_static(const double *z, double *ln_z, double *sin_2piz, double *cos_2piz, uint64_t n);

/* Use this CUDA stream (a cudaStream_t passed as void*) for all later work of the context. */
int mcrt_set_stream(mcrt_ctx *ctx, void *cuda_stream);

/* Launch configuration the transport kernel will use on this device (blocks, threads, dynamic smem). */
int mcrt_launch_config(mcrt_ctx *ctx, int *grid_blocks, int *block_threads, size_t *smem_bytes);

const char *mcrt_last_error(const mcrt_ctx *ctx); /* ctx may be NULL: error of the last failed create */
const char *mcrt_version(void);
void mcrt_destroy(mcrt_ctx *ctx);

#ifdef __cplusplus
}
#endif
#endif /* MCRT_H_ */

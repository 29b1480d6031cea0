/*
 * gcmcrt.h -- C-ABI of libgcmcrt.so: the B200-native (sm_100a) hot path of gCMCRT
 * (Lee et al., arXiv 2110.15640; citations below are /root/reference/PAPER.md line numbers).
 *
 * What the library computes: Monte Carlo photon-packet transport through a 3D spherical-polar
 * atmosphere (radius shells x colatitude cones x longitude half-planes) with
 * next-event estimation ("peel-off", Sect. 4.6, Eq. 14) toward one or more observers, for
 * scattered-light (albedo, Sect. 5.2) and thermal-emission (Sect. 5.3) spectra, per wavelength or
 * correlated-k g-ordinate ("channel").  Every step runs in hand-written CUDA kernels; there is no
 * CPU fallback: without a CUDA device every entry point that needs one returns GCMCRT_E_CUDA.
 *
 * Conventions
 *  - SI units: m, K, kg m^-3, m^2 kg^-1, rad, m/s.  Colatitude theta from +z, longitude phi from +x.
 *  - Cell-flat layout of every per-cell array: [nlon][nlat][nlev], the radial index fastest.
 *    Per-channel tables are [n_chan][nlon][nlat][nlev] (wavelength-major).
 *  - POINTERS: every array argument documented "host|device" may live in host memory (pageable or
 *    pinned) or in device memory; the library asks cudaPointerGetAttributes and copies host arrays
 *    to / from internal device buffers with cudaMemcpyAsync on the caller's stream.  Arguments
 *    documented "host" are read on the CPU during the call.
 *  - OWNERSHIP: the library copies everything it needs during the call that receives it, EXCEPT
 *    DEVICE-resident per-cell opacity tables given to gcmcrt_set_opacity / gcmcrt_set_opacity_nodes
 *    (k_abs, k_sca_ray, k_sca_cld, g_cld): those are borrowed until the next
 *    gcmcrt_set_opacity* / gcmcrt_destroy, because the packed per-cell records are staged from them
 *    by the runs (once for an unshifted run, once per observer with doppler_on, Eq. 33-34).  Host
 *    tables are copied to internal device buffers during the call.  Output buffers are caller-owned.
 *  - STREAMS: all work is enqueued on `stream` (a cudaStream_t passed as void*, NULL = legacy
 *    default stream) and the calls return without waiting for the device: a run's pass loop (fresh
 *    packets -> events -> peel-off, repeated until every packet has ended) is a conditional WHILE
 *    node of a CUDA graph whose bookkeeping runs in device memory.  Results in DEVICE memory
 *    (gcmcrt_result pointers, counters included) are complete when the stream has drained; an
 *    output pointer in HOST memory is filled by a copy at the end of the call followed by ONE
 *    stream synchronisation.  The other places that wait for the device: gcmcrt_grid_create,
 *    gcmcrt_destroy, a run with run_params.timing = 1 (profiling), the test-only gcmcrt_debug_*
 *    calls, lambda given in device memory, and cudaMalloc / cudaFree when an internal buffer has
 *    to grow (first call, or a larger run than any before on the handle).
 *    A run may be issued while `stream` is being captured (cudaStreamBeginCapture): its work,
 *    loop included, becomes part of the caller's graph.  Requirements then: every buffer exists
 *    already (one earlier run of the same size on the handle), all outputs are device memory,
 *    timing = 0, and the capture mode permits cudaStreamBeginCaptureToGraph on an internal stream
 *    (cudaStreamCaptureModeRelaxed or thread-local).
 *  - ENVIRONMENT (read once per handle, for tests and tuning experiments; unset = defaults):
 *    GCMCRT_EVENT_CAP=<n> fixes the event-buffer capacity in records (default: 4 per packet of the
 *    run, 1 Mi .. 128 Mi); GCMCRT_TUNE="a,b,c,d" = lanes waiting before the persistent kernel
 *    serves them (16), lanes parked at a cone / half-plane before a warp serves them (1), wavefront
 *    generations per pass (8; 0 = persistent kernel only), first-pass batch divisor (4).  Neither
 *    changes any result beyond the summation order.  GCMCRT_HOST_LOOP=1 makes the host drive the
 *    pass loop (one wait per pass, no events): profilers (ncu) do not list kernels that run inside
 *    a conditional graph node, so profile with this or with run_params.timing = 1.
 *  - ERRORS: every function returns 0 on success or a negative gcmcrt_status; nothing throws or
 *    exits.  gcmcrt_last_error() returns a static, human-readable description of the last failure
 *    on that handle (or of the last failed gcmcrt_grid_create when passed NULL).
 *  - THREADS: one handle is not thread-safe; distinct handles are independent.
 */
#ifndef GCMCRT_H
#define GCMCRT_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct gcmcrt_grid gcmcrt_grid;

typedef enum gcmcrt_status {
    GCMCRT_OK = 0,
    GCMCRT_E_INVALID = -1, /* bad argument (NULL, non-monotonic edges, sizes <= 0, ...) */
    GCMCRT_E_NOMEM = -2,   /* host or device allocation failed */
    GCMCRT_E_CUDA = -3,    /* a CUDA runtime call or kernel failed, or no device */
    GCMCRT_E_STATE = -4    /* call order: run before set_opacity, ... */
} gcmcrt_status;

/* Run parameters (every default in parentheses is what 0 selects). */
typedef struct gcmcrt_run_params {
    double star_dir[3];          /* unit vector planet -> star (albedo launch) */
    int n_obs;                   /* number of observer directions (>= 0) */
    const double *obs_dir;       /* host [n_obs][3] unit vectors planet -> observer (L326-328) */
    uint64_t packets_per_channel;/* N: normalisation and batch definition */
    uint64_t pkt_begin, pkt_end; /* simulate packet ids [pkt_begin, pkt_end) of [0, N); pkt_end = 0 -> N */
    uint64_t seed;               /* Philox counter words 2,3 */
    int chan_begin, chan_end;    /* channels (local indices of the current table) to run; chan_end = 0 -> all */
    int max_events;              /* stop a packet after this many interactions (0 = unlimited) */
    int scatter_on;              /* 0: only the first peel-off point of each packet (L210, L301) */
    int doppler_on;              /* 1: per-observer Doppler-shifted k_abs (Eq. 33-34), one run per observer */
    int doppler_halfwidth;       /* W: shift clamped to +-W wavelength points (moving window, L403) */
    double emission_bias;        /* xi of the composite emission bias (Sect. 4.3; 0 = unbiased Eq. 13) */
    double tau_vert_max;         /* emission depth cut (L210); <= 0 disables */
    double tau_cut;              /* peel-off contributions with tau_obs > tau_cut are dropped (0 -> 50) */
    int npix;                    /* image side (0 = no images) */
    int n_batches;               /* batches for the batch-means sigma (0 -> 32, max 64) */
    /* Variance reduction (Sect. 4.4-4.5); all 0 = analog transport (L192) */
    int survival_bias;           /* 1: a medium interaction always scatters and W <- W omega (L192-196); the surface
                                    stays analog */
    double roulette_w_min;       /* Russian roulette (L200): when W < roulette_w_min after an interaction ... */
    double roulette_survive;     /* ... the packet survives with this probability and W <- W / roulette_survive
                                    (the paper states neither value; 0 disables).  Requires survival_bias. */
    /* Transmission (Sect. 5.1.1): stellar disc behind the planet for the limb-darkening weight, Eq. 22-23 */
    double star_radius;          /* R_star in m; 0 = no limb darkening (W = 1) */
    double planet_xy[2];         /* sky-plane position of the planet centre relative to the stellar disc centre, m, in
                                    the observer's image frame (e_x = z^ x o^ normalised, e_y = o^ x e_x) */
    double ld_c1, ld_c2;         /* quadratic law I(mu)/I(0) = 1 - c1 (1 - mu) - c2 (1 - mu)^2 (Eq. 22) */
    int cloud_phase;             /* phase function of the cloud scatterers: 0 = Henyey-Greenstein (Eq. 7-8), 1 = two-term
                                    HG (Eq. 10) with the paper's default g1 = g, g2 = -g/2, alpha = 1 - g2^2 (L157),
                                    2 = Draine (Eq. 9) with alpha = 0.5 (L146) and G chosen so that <cos> = g_cld; its
                                    cosine is the zeta-quantile of Eq. 9 (one draw) */
    int forced_scatter;          /* Sect. 4.2 (L179), forced scattering: the optical depth tau_edge along the flight's ray to
                                    where it leaves the grid is integrated first, the flight is drawn as
                                    tau = -ln(1 - zeta (1 - e^-tau_edge)) and the weight is multiplied by 1 - e^-tau_edge;
                                    W e^-tau_edge is added to counters.escaped_weight when the ray leaves through the top.
                                    Rays that end on a reflecting lower boundary stay analog.  1 = the first flight of
                                    albedo packets only ("forced first scattering"); 2 = every flight, albedo and emission
                                    (needs max_events > 0 or Russian roulette to end the packets); excludes
                                    continuous_absorption. */
    int continuous_absorption;   /* Sect. 4.1, Eq. 12: flights are sampled against the scattering extinction only and the
                                    weight decays as W <- W e^-tau_abs over every flight (tau_abs integrated along the
                                    same path); every interaction in the medium is a scattering (no absorption draw, no
                                    omega in the peel-off weight).  Packets end by escaping, at the lower boundary, at
                                    max_events, or by Russian roulette (survival_bias = 1 with roulette_w_min > 0).
                                    Runs through the persistent transport kernel; excludes forced_scatter. */
    double star_solid_angle;     /* Transmission with multiple scattering (Sect. 5.1): with scatter_on and a value > 0 the
                                    packets go on from their chords' starts and scatter; every event's peel-off toward the
                                    observer, W omega Theta e^-tau_obs per steradian, times this solid angle [sr] of the stellar
                                    disc seen from the planet (pi (R_star / a)^2: within it scattered light still reaches
                                    the observer as starlight) is taken off the chord's term of Eq. 21.  0: raytracer mode. */
    double stretch_alpha;        /* Sect. 4.2 (L179), path length stretching (weights of Baes et al. 2016): a in (0, 1) draws
                                    every flight from the stretched law a e^{-a tau} instead of e^{-tau} and multiplies the
                                    weight by the ratio of the two laws for what happened: e^{-(1-a) tau} / a at an interaction
                                    after tau, e^{-(1-a) tau_edge} when the flight leaves the medium or reaches the lower
                                    boundary after tau_edge.  With forced_scatter (1: first flight, 2: every flight) the hybrid
                                    scheme: the stretched law truncated at tau_edge, tau = -ln(1 - zeta (1 - e^{-a tau_edge})) / a,
                                    extra weight factor 1 - e^{-a tau_edge}.  0 or 1 = off.  Excludes continuous_absorption. */
    int timing;                  /* 0: the run is only enqueued (see STREAMS); the ms_* counters stay 0.
                                    1: profiling run -- the pass loop is driven by the host, which waits for every pass
                                    and records cudaEvents around its kernels to fill the ms_* counters */
    int concurrency;             /* K = 2 .. 8: the channels of the run (independent, L79) are cut into K contiguous parts that
                                    run side by side -- part 0 on this handle and the caller's stream, the others on internal
                                    copies of the grid handle with working buffers of their own (they borrow this handle's
                                    opacity tables) and internal streams that fork from the caller's stream and join it before
                                    the call's results are complete -- so that the kernels of one part use the issue slots and
                                    memory latencies another leaves idle.  Same results (packets are keyed by channel and
                                    index); counters are summed over the parts.  The internal handles are created by the
                                    first such call, which waits for the device; working memory grows K-fold.  Every part
                                    stages the tables (per observer with doppler_on), and builds the emission CDF, of its own
                                    channels only, so the parts repeat no work.  0 or 1, and whenever it does not apply
                                    (timing = 1, transmission, fewer than K channels in the run, a stream that is being
                                    captured, GCMCRT_HOST_LOOP): one run on this handle. */
} gcmcrt_run_params;

typedef struct gcmcrt_counters {
    uint64_t events;             /* peel-off points (emission launches, interactions, surface hits) */
    uint64_t segments_transport; /* cell crossings on packet flights */
    uint64_t segments_peel;      /* cell crossings on peel-off rays */
    uint64_t packets_escaped, packets_absorbed, packets_surface, packets_stuck;
    double escaped_weight;
    uint64_t passes;             /* transport/peel kernel pairs launched */
    uint64_t rays_peel;          /* peel-off rays integrated */
    uint64_t launches;           /* kernels this call launched (all kinds) */
    /* device time of this call's kernels by kind, from cudaEvents recorded on the caller's stream around each
       launch (milliseconds, summed over passes / observers); filled by runs with run_params.timing = 1, else 0 */
    double ms_stage, ms_emission_cdf, ms_transport, ms_peel;
    double ms_sort;              /* counting sort of the event records by (channel, cell) before each peel pass */
    uint64_t device_status;      /* 0 = the pass loop ran to its end; 1 = suspended-packet list overflow, 2 = pass limit
                                    reached (both "cannot happen": the library sizes its buffers so); with host-resident
                                    counters a non-zero value also makes the call return GCMCRT_E_CUDA */
} gcmcrt_counters;

/* Output buffers, all caller-owned, host|device, nullable unless stated. */
typedef struct gcmcrt_result {
    double *flux_sum;      /* REQUIRED [n_chan_run][n_obs][n_batches]: raw sums of f (Eq. 14) */
    double *L_tot;         /* [n_chan_run][n_obs]: total luminosity (Eq. 27-28), emission only */
    double *value;         /* [n_chan_run][n_obs]: albedo: reflected fraction per steradian S/N (A_g = pi*value at
                              zero phase, Eq. 24); emission: L_p = L_tot S/N in W m^-1 sr^-1 (Eq. 28) */
    double *sigma;         /* [n_chan_run][n_obs]: batch-means standard error of value */
    float *image;          /* [n_chan_run][n_obs][npix][npix] (L83) */
    uint32_t *event_count; /* [n_chan_run][pkt_end-pkt_begin]: peel-off points per packet */
    gcmcrt_counters *counters; /* one struct, host|device (device: assembled by a kernel, no host wait) */
    float *contrib;        /* [n_chan_run][n_obs][2][ncell] (cell-flat layout): contribution functions of Sect. 6,
                              Eq. 32, as raw sums of the peeled-off f per event cell: [0] thermal (emission points),
                              [1] scattered (medium and surface events).  CF = contrib / sum over cells. */
} gcmcrt_result;

/*
 * gcmcrt_grid_create -- build the 3D spherical grid (D1, D2, D4, D5) and stage its
 * geometry tables on the current CUDA device.
 *   r_edges[nlev+1]     host, strictly ascending; r_edges[0] = lower boundary R_p0, last = R_TOA
 *   colat_edges[nlat+1] host, ascending, must span 0..pi   (nlat = 1: no cones at all)
 *   lon_edges[nlon+1]   host, ascending, must span 0..2pi  (nlon = 1: no half-planes)
 *   T, rho              host|device [nlon][nlat][nlev] (copied)
 *   u, v, w             host|device, same layout, nullable (east, north, up wind; Eq. 33), copied
 *   Omega               rotation rate (Eq. 33)
 *   surface_albedo      Lambert albedo of the lower boundary (Eq. 3-4); 0 = absorbing
 * Errors: E_INVALID (NULL, sizes, non-monotonic), E_NOMEM, E_CUDA.  *out is NULL on failure.
 */
int gcmcrt_grid_create(gcmcrt_grid **out, int nlev, int nlat, int nlon,
                       const double *r_edges, const double *colat_edges, const double *lon_edges,
                       const float *T, const float *rho,
                       const float *u, const float *v, const float *w, double Omega,
                       float surface_albedo, void *stream);

/*
 * gcmcrt_set_opacity -- give the per-channel, per-cell opacities (D3) of
 * channels chan0 .. chan0+n_chan-1.  The packed records alpha_ext = rho (k_abs + k_ray + k_cld), omega, P_gas
 * (Eq. 11) and g per (channel, cell) (A0) are staged from them by the first run that needs them (an unshifted run
 * stages once; a doppler_on run stages per observer; a continuous_absorption run stages its own variant).  chan0 is
 * the global index of the first channel: it keys the random streams, so results do not depend on how a long table
 * is cut into batches.
 *   lambda[n_chan]  host, m (Planck function, Doppler spacing)
 *   k_abs           host|device [n_chan][nlon][nlat][nlev], required
 *   k_sca_ray       host|device, nullable (= 0): Rayleigh scattering opacity
 *   k_sca_cld       host|device, nullable (= 0): cloud scattering opacity
 *   g_cld           host|device, nullable (= 0): asymmetry parameter of the cloud scatterers
 *   (device-resident tables are borrowed until the next gcmcrt_set_opacity* / gcmcrt_destroy, see OWNERSHIP above)
 * Errors: E_INVALID, E_NOMEM, E_CUDA.
 */
int gcmcrt_set_opacity(gcmcrt_grid *grid, int chan0, int n_chan, const float *lambda,
                       const float *k_abs, const float *k_sca_ray, const float *k_sca_cld,
                       const float *g_cld, void *stream);

/*
 * gcmcrt_set_opacity_nodes -- as gcmcrt_set_opacity, but the absorption opacity comes from (T, log10 p) node tables
 * and is interpolated to the cells on the device (the GPU opacity interpolation the paper plans, Sect. 7; its
 * stated bottleneck is reading per-cell 3D opacity tables): a channel costs nT*nP floats instead of ncell.
 *   k_abs(c, cell) = bilinear interpolation of node_kabs[c][nT][nP] at (T[cell], log10 p_cell[cell]), clamped to the
 *   table; with doppler_on the shifted opacity (Eq. 34) interpolates between the bilinear values of the two
 *   neighbouring channels.
 *   node_kabs   host|device [n_chan][nT][nP] m^2/kg (copied)
 *   T_nodes     host [nT] K, uniformly spaced ascending;  logp_nodes  host [nP] log10(Pa), uniformly spaced ascending
 *   p_cell      host|device [nlon][nlat][nlev] Pa (copied)
 *   lambda, k_sca_ray, k_sca_cld, g_cld: as gcmcrt_set_opacity (per-cell tables, nullable)
 * Errors: E_INVALID, E_NOMEM, E_CUDA.
 */
int gcmcrt_set_opacity_nodes(gcmcrt_grid *grid, int chan0, int n_chan, const float *lambda,
                             const float *node_kabs, int nT, int nP, const float *T_nodes, const float *logp_nodes,
                             const float *p_cell, const float *k_sca_ray, const float *k_sca_cld,
                             const float *g_cld, void *stream);

/*
 * gcmcrt_run_albedo -- scattered-light run (Sect. 5.2): packets enter uniformly over the star-facing TOA disc
 * (incident flux normalised to 1, L283), fly sampled optical depths (L192), peel off to every observer at every
 * interaction (Eq. 14), scatter with Rayleigh (Eq. 5-6) / Henyey-Greenstein (Eq. 7-8) chosen by P_gas (Eq. 11)
 * or are absorbed (L192).
 * gcmcrt_run_emission -- thermal run (Sect. 5.3): packets are emitted from cells in proportion to their
 * luminosity (Eq. 13, Eq. 27; composite bias xi), peel off at the emission point (L210) and, if scatter_on,
 * continue as above.  value = L_tot/N sum f (Eq. 28).
 * Errors: E_STATE (no opacity set), E_INVALID, E_NOMEM, E_CUDA.
 */
int gcmcrt_run_albedo(gcmcrt_grid *grid, const gcmcrt_run_params *params, gcmcrt_result *out, void *stream);
int gcmcrt_run_emission(gcmcrt_grid *grid, const gcmcrt_run_params *params, gcmcrt_result *out, void *stream);

/*
 * gcmcrt_run_transmission -- transmission spectrum by random transit chords (Sect. 5.1, Eq. 20-21): the "raytracer
 * scheme with random transit chord sampler" of L261, or -- with scatter_on and star_solid_angle > 0 -- the scheme with
 * multiple scattering of L259 (the paper describes it in words; reading N12): chord i then contributes
 * W_i b_i [1 - exp(-tau_i) - star_solid_angle * sum over the packet's events of W omega Theta exp(-tau_obs)].  Packet i of a channel draws an impact parameter b_i uniform in [R_p0, R_TOA] and an
 * azimuth around the limb; tau_i is the extinction optical depth of the whole chord along obs_dir (planet -> observer)
 * -- with doppler_on through that observer's Doppler-shifted table (Eq. 33-34, the set-up of the paper's Sect. 13).
 *   flux_sum[c][o][batch] = sum_i W_i [1 - exp(-tau_i)] b_i      (W_i: limb darkening, Eq. 22-23; 1 if star_radius = 0)
 *   value[c][o] = <I_p> = (R_TOA - R_p0) / N * sum  [m^2] (Eq. 21), sigma its batch-means standard error;
 *   the caller forms (R_p / R_star)^2 = (R_p0^2 + 2 <I_p>) / R_star^2 (Eq. 20).
 * star_dir, emission_bias, npix, image, contrib are not used; scatter_on, max_events, the variance-reduction switches and
 * event_count (interactions per packet, first observer's run) only with multiple scattering.  n_obs >= 1.
 * Errors: as gcmcrt_run_albedo.
 */
int gcmcrt_run_transmission(gcmcrt_grid *grid, const gcmcrt_run_params *params, gcmcrt_result *out, void *stream);

/* gcmcrt_destroy -- synchronise the device, free everything the handle owns.  NULL is a no-op. */
int gcmcrt_destroy(gcmcrt_grid *grid);

/* Text of the last error on this handle (NULL: last failed gcmcrt_grid_create).  Never NULL. */
const char *gcmcrt_last_error(const gcmcrt_grid *grid);

/*
 * gcmcrt_debug_ray_tau -- test-only: optical depth of channel `chan` (local index) from pos[m] along dir[m] to
 * the TOA with the peel-off ray integrator (A7), without a run.  hit_surface[m] = 1 when the ray ends on the
 * lower boundary (tau then is the depth down to it).  The ray runs through the table staged last: the unshifted one
 * (staged by this call if no run has staged anything yet), or the Doppler table of the last doppler_on run's observer.
 *   pos, dir  host|device [n][3] float; tau host|device [n] float; hit_surface host|device [n] int (nullable)
 */
int gcmcrt_debug_ray_tau(gcmcrt_grid *grid, int chan, long n, const float *pos, const float *dir,
                         float *tau, int *hit_surface, void *stream);

/*
 * gcmcrt_debug_philox -- test-only: out[m][4] = Philox4x32-10(counter = ctr[m][4], key = key[m][2]) computed on
 * the device by the generator the packet kernels use (A3); all arrays host|device.
 */
int gcmcrt_debug_philox(long n, const uint32_t *ctr, const uint32_t *key, uint32_t *out, void *stream);

/*
 * gcmcrt_emission_ltot_static -- the total luminosities L_tot[c] (Eq. 27 summed over the cells, with the depth cut of
 * L210; the normalisation of Eq. 28) of channels chan_begin .. chan_end-1 (chan_end = 0: to the end of the table) of the
 * tables that are staged on the handle, computed WITHOUT ANY ALLOCATION: for callers that must not reach cudaMalloc (code
 * under stream capture, tight serving loops, harnesses that forbid it).  The same arithmetic in the same order as the
 * L_tot output of gcmcrt_run_emission (which keeps its per-column totals in a buffer of the handle that grows on demand);
 * here they live in a file-scope device array of GCMCRT_STATIC_SCRATCH_BYTES that every GPU which loads the library
 * holds until the process exits.
 *   L_tot[chan_end - chan_begin]  host|device.  Device: the call only enqueues two kernels on `stream`.  Host: the result
 *                                 is copied from the array and the call waits for the stream.
 *   tau_vert_max                  as run_params.tau_vert_max (<= 0: no depth cut)
 * The tables must be staged already -- by any run on this handle after the last gcmcrt_set_opacity* (a doppler_on run
 * leaves its last observer's shifted table: that is then the table L_tot is of) -- because staging may allocate; E_STATE
 * otherwise, and when a run_params.concurrency run left only a part of the channels staged on this handle.
 * LIMIT: (n_channels * nlat * nlon + n_channels) * 8 bytes <= GCMCRT_STATIC_SCRATCH_BYTES, else E_INVALID with a message
 * that states both sizes -- pass fewer channels per call (cfg2's 64 x 32 columns: 511 channels; cfg5's 128 x 64: 127).
 * SHARED STATE: every call on a device uses the same array, which keeps the last call's contents (nothing in it has to
 * start at zero: a call writes every entry before it reads it).  Calls that overlap on the GPU -- different streams, or
 * different handles or host threads without an ordering between them -- race; calls on one stream are safe.
 * Calls no cudaMalloc / cudaFree and no allocating library routine.  Errors: E_INVALID, E_STATE, E_CUDA.
 */
#define GCMCRT_STATIC_SCRATCH_BYTES (8u << 20)
int gcmcrt_emission_ltot_static(gcmcrt_grid *grid, int chan_begin, int chan_end, double tau_vert_max, double *L_tot,
                                void *stream);

/* Library build information: "gcmcrt <version> sm_100a ..." */
const char *gcmcrt_version(void);

#ifdef __cplusplus
}
#endif
#endif /* GCMCRT_H */

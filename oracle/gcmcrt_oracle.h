/*
 * gcmcrt_oracle.h -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, serial, fp64 CPU restatement of the hot path of gCMCRT
 * (arXiv 2110.15640; /root/reference/PAPER.md): Monte Carlo photon-packet
 * transport with next-event estimation ("peel-off") for albedo and emission
 * spectra on a 3D spherical-polar grid.  It follows the paper step by step in
 * the paper's order (citations are "PAPER.md:Lnnn, section/equation") and the
 * readings C1..C20 of SURVEY.md section 8(c), restated in DESIGN.md.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference leg may build, load or call this.  It shares no code,
 * header, table or constant generator with paper_2110_15640_b200/ (the CUDA
 * path) and neither imports the other.
 *
 * Pins (tests/test_oracle_*.py, all `-m "not gpu"`): Philox known-answer
 * vectors; closed-form CDFs and moments of every phase-function sampler;
 * analytic chord optical depths; grid-refinement invariance; e^{-tau}
 * transmission; Lambert sphere 2/3 and its phase law; exact Chandrasekhar
 * H-function albedos; isothermal emitter chord integral; energy conservation;
 * peel-off <-> escape consistency; brute-force enumeration on a 1-cell grid;
 * rotational invariance; Eq. 33 vector identity; the image frame (C19) by the
 * brightness law of a Lambert sphere and the lit half at quadrature; path
 * length stretching and its hybrid by the exact albedos and analog agreement.
 * The whole library also runs under ASan + UBSan (tests/test_oracle_sanitizers.py).
 * Paper-printed numeric values: none exist (Fig. 1 is an image) -> "parity
 * against paper-printed values: unpinned"; every function is pinned by the
 * closed forms above instead.
 */
#ifndef GCMCRT_ORACLE_H
#define GCMCRT_ORACLE_H
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* D1/D2/D4/D5: the 3D spherical grid and
 * its per-cell fields, cell-flat index = (k*nlat + j)*nlev + i with i the
 * radial (fastest) index, j colatitude, k longitude. */
typedef struct {
    int nlev, nlat, nlon;
    const double *r_edges;     /* [nlev+1] ascending, m; [0]=R_p0, [nlev]=R_TOA */
    const double *colat_edges; /* [nlat+1] 0..pi */
    const double *lon_edges;   /* [nlon+1] 0..2pi */
    const float *T;            /* [ncell] K */
    const float *rho;          /* [ncell] kg m^-3 */
    const float *u, *v, *w;    /* [ncell] m/s east, north, up; nullable */
    double Omega;              /* rad/s */
    double surface_albedo;     /* 0 = absorbing lower boundary (C5) */
} orc_grid;

/* D3: per channel, per cell opacities. */
typedef struct {
    int n_chan;
    int chan0;               /* global index of the first channel (Philox key) */
    const float *lambda;     /* [n_chan] m */
    const float *k_abs;      /* [n_chan][ncell] m^2/kg */
    const float *k_sca_ray;  /* nullable */
    const float *k_sca_cld;  /* nullable */
    const float *g_cld;      /* nullable -> 0 */
} orc_opacity;

typedef struct {
    double star_dir[3];
    int n_obs;
    const double *obs_dir;   /* [n_obs][3] unit vectors */
    uint64_t packets_per_channel; /* N: defines batches and normalisation */
    uint64_t pkt_begin, pkt_end;  /* packet ids simulated, [begin,end) within [0,N) */
    uint64_t seed;
    int max_events;          /* 0 = unlimited */
    int scatter_on;
    int doppler_on;
    int doppler_halfwidth;   /* W, in wavelength points */
    double emission_bias;    /* xi (C10) */
    double tau_vert_max;     /* <=0: no cut (L210) */
    double tau_cut;          /* peel-off contributions with tau_obs > tau_cut are 0 */
    int npix;                /* 0 = no images */
    int n_batches;
    int n_threads;           /* OpenMP threads over batches; <=1 serial */
    /* Variance reduction (Sect. 4.4-4.5); all 0 = analog transport */
    int survival_bias;       /* 1: a medium interaction always scatters and W <- W omega (L192-196) */
    double roulette_w_min;   /* Russian roulette (L200) when W < roulette_w_min after an interaction ... */
    double roulette_survive; /* ... the packet survives with this probability and W <- W / roulette_survive */
    /* Transmission (Sect. 5.1): stellar disc for the limb-darkening weight of Eq. 22-23; star_radius = 0: W = 1 */
    double star_radius;      /* R_star, m */
    double planet_xy[2];     /* sky-plane position of the planet centre relative to the stellar disc centre, m, in
                                the observer's image frame (C19: e_x = z^ x o^ normalised, e_y = o^ x e_x) */
    double ld_c1, ld_c2;     /* quadratic limb-darkening law, Eq. 22 */
    int cloud_phase;         /* cloud scatterers: 0 = HG (Eq. 7-8), 2 = Draine (Eq. 9, alpha = 0.5), 1 = two-term HG (Eq. 10) with the paper's default
                                g1 = g, g2 = -g/2, alpha = 1 - g2^2 (L157) */
    int forced_scatter;      /* Sect. 4.2 (L179; Cashwell & Everett 1959): 1 = forced first scattering of albedo packets: the
                                first flight must end inside the grid: tau_edge = optical depth along the launch ray to
                                where it leaves the grid (the extra ray trace of L179), tau = -ln(1 - zeta (1 - e^-tau_edge)),
                                W = 1 - e^-tau_edge.  2 = the same at every flight (albedo and emission).  Rays that
                                end on a reflecting lower boundary stay analog. */
    int continuous_absorption; /* Sect. 4.1, Eq. 12: flights are sampled against the scattering extinction only and the
                                weight decays as W <- W e^-tau_abs along every flight; every interaction in the medium
                                is then a scattering (no absorption draw, no omega in the peel-off weight) */
    double star_solid_angle; /* Sect. 5.1, L259 (reading N12): > 0 with scatter_on switches multiple scattering on in
                                transmission: solid angle [sr] of the stellar disc seen from the planet, over which light
                                scattered back toward the observer still counts as transmitted starlight */
    double stretch_alpha;    /* Sect. 4.2 (L179; Baes et al. 2016), path length stretching: flights are drawn from
                                a e^{-a tau} with a = stretch_alpha in (0, 1) and weighted by p / q (0 or 1: off).  With
                                forced_scatter: the hybrid scheme, the stretched law truncated at tau_edge */
} orc_params;

typedef struct {
    uint64_t events;             /* peel-off points */
    uint64_t segments_transport; /* cell crossings on flights */
    uint64_t segments_peel;      /* cell crossings on peel-off rays */
    uint64_t packets_escaped, packets_absorbed, packets_surface, packets_stuck;
    double escaped_weight;
} orc_counters;

typedef struct {
    double *flux_sum;      /* [n_chan][n_obs][n_batches] raw sums of f (Eq. 14) */
    double *L_tot;         /* [n_chan] (emission; with doppler_on [n_chan][n_obs]) */
    double *image;         /* nullable [n_chan][n_obs][npix][npix] */
    uint32_t *event_count; /* nullable [n_chan][N] */
    orc_counters counters;
    double *contrib;       /* nullable [n_chan][n_obs][2][ncell]: Eq. 32 numerators: peeled-off f summed per event
                              cell, [0] thermal (emission points), [1] scattered (medium + surface events) */
} orc_result;

/* A3: Philox4x32-10 (Salmon et al. 2011), C2. */
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]);
/* C2: zeta = ((u>>9)+0.5) * 2^-23 (exact in fp32 and fp64) */
double orc_u32_to_zeta(uint32_t u);
/* The block of four zetas for (seed, channel, packet, event, purpose). */
void orc_zeta_block(uint64_t seed, uint32_t chan, uint32_t pkt, uint32_t event, uint32_t purpose, double z[4]);

/* Phase-function samplers (Eq. 2, 4, 6 [C7], 8 [C8]) and densities per steradian. */
double orc_sample_isotropic(double zeta);
double orc_sample_lambert(double zeta);
double orc_sample_rayleigh(double zeta);
double orc_sample_hg(double g, double zeta);
double orc_phase_rayleigh(double mu);
double orc_phase_hg(double g, double mu);
/* Eq. 10 with g1 = g, g2 = -g/2, alpha = 1 - g2^2 (L157); zeta_lobe < alpha picks the forward lobe (L152) */
double orc_sample_tthg(double g, double zeta_lobe, double zeta);
double orc_phase_tthg(double g, double mu);
double orc_draine_G(double g);                 /* Eq. 9: G with <cos> = g at alpha = 0.5 */
double orc_phase_draine(double g, double mu);
double orc_sample_draine(double g, double zeta);
/* C9: rotate unit vector n by polar angle acos(ct) and azimuth psi. */
void orc_rotate(const double n[3], double ct, double psi, double out[3]);

/* O1: cell volume. */
double orc_cell_volume(const orc_grid *g, int i, int j, int k);
/* Locate (i,j,k) of a point (used for launch and for debug rays). */
void orc_locate(const orc_grid *g, const double p[3], int ijk[3]);
/* B_lambda(T), SI (W m^-3 sr^-1). */
double orc_planck(double lambda, double T);
/* O9 / Eq. 33: line-of-sight velocity, both the paper's trigonometric form and the vector form. */
double orc_vlos_eq33(double u, double v, double w, double Omega, double r, double theta, double phi,
                     double theta_v, double phi_v);
double orc_vlos_vector(double u, double v, double w, double Omega, double r, double theta, double phi,
                       const double obs[3]);

/* O5: optical depth from p along dir to the TOA for channel `chan` (local index)
 * (observer index obs_index selects the Doppler table; -1 = unshifted).
 * hit_surface[m]=1 if the ray ends on the lower boundary.  nseg/path optional. */
int orc_ray_tau(const orc_grid *g, const orc_opacity *op, int chan, long n,
                const double *pos, const double *dir, double *tau, int *hit_surface,
                long *nseg, double *path_len);

/* O2: staged per-cell quantities of one channel (for tests): alpha_ext, omega, pgas, g, L_i, cdf. */
int orc_channel_prep(const orc_grid *g, const orc_opacity *op, const orc_params *prm, int chan, int obs_index,
                     double *alpha, double *omega, double *pgas, double *gg, double *L_cell, double *L_tot);

/* The two drivers (section 3 call stacks). */
int orc_run_albedo(const orc_grid *g, const orc_opacity *op, const orc_params *prm, orc_result *out);
int orc_run_emission(const orc_grid *g, const orc_opacity *op, const orc_params *prm, orc_result *out);
/* Transmission spectrum by random transit chords (Sect. 5.1, Eq. 20-21).  Multiple scattering off (L261: "reduces the
 * model to a raytracer scheme with random transit chord sampler"): flux_sum[c][o][batch] = sum over packets of
 * W [1 - exp(-tau_i)] b_i; <I_p> = (R_TOA - R_p0) / N * sum (Eq. 21); W from Eq. 22-23.  With scatter_on and
 * star_solid_angle > 0 the packets go on to scatter (L259) and every event's peel-off toward the observer, times the
 * stellar solid angle, is taken off the chord's term (reading N12 in DESIGN.md). */
int orc_run_transmission(const orc_grid *g, const orc_opacity *op, const orc_params *prm, orc_result *out);

#ifdef __cplusplus
}
#endif
#endif

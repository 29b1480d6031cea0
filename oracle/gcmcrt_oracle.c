/*
 * gcmcrt_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE (see gcmcrt_oracle.h).
 *
 * Serial fp64 restatement of gCMCRT's packet transport + peel-off, following
 * /root/reference/PAPER.md in the paper's order.  Where the paper is silent the
 * reading taken is the one listed in DESIGN.md ("Readings", C1..C20).
 * No blocking, fusion or reordering: every segment recomputes all six face
 * distances from the current position (O5), every event peels to every
 * observer with a full ray integral (Eq. 14).
 */
#include "gcmcrt_oracle.h"

#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define PI 3.14159265358979323846
#define H_PLANCK 6.62607015e-34
#define C_LIGHT 299792458.0
#define K_BOLTZ 1.380649e-23

/* ------------------------------------------------------------------ */
/* A3 / C2: Philox4x32-10 (Salmon, Moraes, Dror, Shaw 2011).           */
/* ------------------------------------------------------------------ */
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        uint64_t p0 = (uint64_t)0xD2511F53u * (uint64_t)c0;
        uint64_t p1 = (uint64_t)0xCD9E8D57u * (uint64_t)c2;
        uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
        uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
        uint32_t n0 = hi1 ^ c1 ^ k0;
        uint32_t n1 = lo1;
        uint32_t n2 = hi0 ^ c3 ^ k1;
        uint32_t n3 = lo0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* C2: zeta = ((u >> 9) + 0.5) 2^-23 in (0,1): 2k+1 < 2^24, so it is exactly representable in fp32 as well as
 * fp64 (the 24-bit variant ((u>>8)+0.5) 2^-24 is not), never 0 or 1; the largest sampled tau is 24 ln 2 = 16.6. */
double orc_u32_to_zeta(uint32_t u)
{
    return ((double)(u >> 9) + 0.5) * (1.0 / 8388608.0);
}

/* C2: key = (channel, packet); counter = (event, purpose, seed_lo, seed_hi). */
void orc_zeta_block(uint64_t seed, uint32_t chan, uint32_t pkt, uint32_t event, uint32_t purpose, double z[4])
{
    uint32_t ctr[4] = { event, purpose, (uint32_t)(seed & 0xffffffffu), (uint32_t)(seed >> 32) };
    uint32_t key[2] = { chan, pkt };
    uint32_t out[4];
    orc_philox4x32_10(ctr, key, out);
    for (int m = 0; m < 4; ++m) z[m] = orc_u32_to_zeta(out[m]);
}

/* ------------------------------------------------------------------ */
/* Section 3: phase functions and their samplers.                      */
/* ------------------------------------------------------------------ */
/* Eq. 2 */
double orc_sample_isotropic(double zeta) { return 2.0 * zeta - 1.0; }
/* Eq. 4 */
double orc_sample_lambert(double zeta) { return sqrt(zeta); }
/* Eq. 6 is garbled as printed; reading C7: the Cardano root of
 * the CDF of Eq. 5, q = 4 zeta - 2, u = cbrt(q + sqrt(1+q^2)), cos = u - 1/u. */
double orc_sample_rayleigh(double zeta)
{
    double q = 4.0 * zeta - 2.0;
    double u = cbrt(q + sqrt(1.0 + q * q));
    return u - 1.0 / u;
}
/* Eq. 8; C8: |g| < 1e-3 -> isotropic (Eq. 2). */
double orc_sample_hg(double g, double zeta)
{
    if (fabs(g) < 1e-3) return 2.0 * zeta - 1.0;
    double t = (1.0 - g * g) / (1.0 - g + 2.0 * g * zeta);
    return (1.0 + g * g - t * t) / (2.0 * g);
}
/* Eq. 5 normalised per steradian: 3(1+mu^2)/(16 pi). */
double orc_phase_rayleigh(double mu) { return 3.0 * (1.0 + mu * mu) / (16.0 * PI); }
/* Eq. 7 normalised per steradian. */
double orc_phase_hg(double g, double mu)
{
    double d = 1.0 + g * g - 2.0 * g * mu;
    return (1.0 - g * g) / (4.0 * PI * d * sqrt(d));
}

/* Eq. 10: two-term HG with the default g1 = g, g2 = -g/2, alpha = 1 - g2^2. */
double orc_phase_tthg(double g, double mu)
{
    const double g2 = -0.5 * g, a = 1.0 - g2 * g2;
    return a * orc_phase_hg(g, mu) + (1.0 - a) * orc_phase_hg(g2, mu);
}
/* L152: zeta_lobe < alpha -> Eq. 8 with g1, else Eq. 8 with g2. */
double orc_sample_tthg(double g, double zeta_lobe, double zeta)
{
    const double g2 = -0.5 * g, a = 1.0 - g2 * g2;
    return zeta_lobe < a ? orc_sample_hg(g, zeta) : orc_sample_hg(g2, zeta);
}

/* Eq. 9: Draine (2003) phase function, alpha = 0.5 by default (L146).  "G(g) is a function of the
 * asymmetry parameter g": the first moment of Eq. 9 is <cos> = G (1 + alpha (3 + 2 G^2) / 5) / (1 + alpha (1 + 2 G^2) / 3)
 * (pinned by quadrature in tests/test_oracle_pins.py); G is the root of <cos>(G) = g in (-1, 1), found by bisection. */
#define DRAINE_ALPHA 0.5
static double draine_first_moment(double G, double a)
{
    return G * (1.0 + a * (3.0 + 2.0 * G * G) / 5.0) / (1.0 + a * (1.0 + 2.0 * G * G) / 3.0);
}
double orc_draine_G(double g)
{
    double lo = -1.0, hi = 1.0;
    for (int it = 0; it < 60; ++it) {
        double mid = 0.5 * (lo + hi);
        if (draine_first_moment(mid, DRAINE_ALPHA) < g) lo = mid; else hi = mid;
    }
    return 0.5 * (lo + hi);
}
/* Eq. 9 per steradian (the printed form integrates to 4 pi over the sphere). */
double orc_phase_draine(double g, double mu)
{
    const double a = DRAINE_ALPHA, G = orc_draine_G(g);
    const double d = 1.0 + G * G - 2.0 * G * mu;
    return (1.0 - G * G) / (1.0 + a * (1.0 + 2.0 * G * G) / 3.0) * (1.0 + a * mu * mu) / (d * sqrt(d)) / (4.0 * PI);
}
/* int_{-1}^{mu} (1 + alpha x^2) (1 + G^2 - 2 G x)^(-3/2) dx, by the substitution t = 1 + G^2 - 2 G x. */
static double draine_cdf_unnormalised(double G, double a, double mu)
{
    if (fabs(G) < 1e-3) return (mu + 1.0) + a * (mu * mu * mu + 1.0) / 3.0;   /* G -> 0: 1 + alpha mu^2 (cf. C8) */
    const double A = 1.0 + G * G, B = 2.0 * G;
    const double c0 = 1.0 + a * A * A / (B * B), c1 = 2.0 * a * A / (B * B), c2 = a / (3.0 * B * B);
    double t = A - B * mu, t0 = A + B;
    double H = (2.0 / B) * (c0 / sqrt(t) + c1 * sqrt(t) - c2 * t * sqrt(t));
    double H0 = (2.0 / B) * (c0 / sqrt(t0) + c1 * sqrt(t0) - c2 * t0 * sqrt(t0));
    return H - H0;
}
/* The paper samples Eq. 9 by the Gibbs scheme of Zhang (2019), which it only cites (L146); here the cosine is the
 * zeta-quantile of Eq. 9 itself (inverse of its closed-form CDF, bisection): the same distribution from one draw,
 * which keeps the one-block-per-event stream layout (reading N10). */
double orc_sample_draine(double g, double zeta)
{
    const double a = DRAINE_ALPHA, G = orc_draine_G(g);
    const double total = draine_cdf_unnormalised(G, a, 1.0);
    double lo = -1.0, hi = 1.0;
    for (int it = 0; it < 60; ++it) {
        double mid = 0.5 * (lo + hi);
        if (draine_cdf_unnormalised(G, a, mid) < zeta * total) lo = mid; else hi = mid;
    }
    return 0.5 * (lo + hi);
}

/* C9: rotate n by polar angle acos(ct) and azimuth psi. */
void orc_rotate(const double n[3], double ct, double psi, double out[3])
{
    double st = sqrt(fmax(0.0, 1.0 - ct * ct));
    double cp = cos(psi), sp = sin(psi);
    double x, y, z;
    double s2 = n[0] * n[0] + n[1] * n[1];   /* sin^2 of n's polar angle, free of cancellation */
    if (s2 < 1e-12) {                        /* within 1e-6 rad of the z axis: use z^ as the axis */
        x = st * cp;
        y = st * sp;
        z = ct * (n[2] >= 0.0 ? 1.0 : -1.0);
    } else {
        double sq = sqrt(s2);
        x = st * (n[0] * n[2] * cp - n[1] * sp) / sq + n[0] * ct;
        y = st * (n[1] * n[2] * cp + n[0] * sp) / sq + n[1] * ct;
        z = -st * cp * sq + n[2] * ct;
    }
    double nn = sqrt(x * x + y * y + z * z);
    out[0] = x / nn; out[1] = y / nn; out[2] = z / nn;
}

/* B_lambda(T) = 2hc^2 lambda^-5 / expm1(hc / (lambda k T)); SI. (Eq. 27's B) */
double orc_planck(double lambda, double T)
{
    double x = H_PLANCK * C_LIGHT / (lambda * K_BOLTZ * T);
    return 2.0 * H_PLANCK * C_LIGHT * C_LIGHT / (lambda * lambda * lambda * lambda * lambda) / expm1(x);
}

/* ------------------------------------------------------------------ */
/* O1: geometry.                                                       */
/* ------------------------------------------------------------------ */
typedef struct {
    int nlev, nlat, nlon, ncell;
    const double *R, *th, *ph;
    double *cth, *sth;  /* cos / sin of colatitude edges */
    double *cph, *sph;  /* cos / sin of longitude edges */
    double Rtoa, s_eps;
    int maxseg;
} geom_t;

static int geom_init(geom_t *G, const orc_grid *g)
{
    G->nlev = g->nlev; G->nlat = g->nlat; G->nlon = g->nlon;
    G->ncell = g->nlev * g->nlat * g->nlon;
    G->R = g->r_edges; G->th = g->colat_edges; G->ph = g->lon_edges;
    G->cth = (double *)malloc(sizeof(double) * (size_t)(g->nlat + 1) * 2);
    G->sth = G->cth + (g->nlat + 1);
    G->cph = (double *)malloc(sizeof(double) * (size_t)(g->nlon + 1) * 2);
    G->sph = G->cph + (g->nlon + 1);
    if (!G->cth || !G->cph) return -1;
    for (int j = 0; j <= g->nlat; ++j) { G->cth[j] = cos(G->th[j]); G->sth[j] = sin(G->th[j]); }
    for (int k = 0; k <= g->nlon; ++k) { G->cph[k] = cos(G->ph[k]); G->sph[k] = sin(G->ph[k]); }
    G->Rtoa = G->R[g->nlev];
    G->s_eps = 1e-9 * G->Rtoa;           /* O5 */
    G->maxseg = 8 * (g->nlev + g->nlat + g->nlon) + 64;
    return 0;
}
static void geom_free(geom_t *G) { free(G->cth); free(G->cph); }

static inline int cell_index(const geom_t *G, int i, int j, int k) { return (k * G->nlat + j) * G->nlev + i; }
static inline double dot3(const double a[3], const double b[3]) { return a[0] * b[0] + a[1] * b[1] + a[2] * b[2]; }

/* O1: V = (R_{i+1}^3 - R_i^3)/3 (cos th_j - cos th_{j+1}) (ph_{k+1} - ph_k) */
double orc_cell_volume(const orc_grid *g, int i, int j, int k)
{
    double r0 = g->r_edges[i], r1 = g->r_edges[i + 1];
    return (r1 * r1 * r1 - r0 * r0 * r0) / 3.0 * (cos(g->colat_edges[j]) - cos(g->colat_edges[j + 1])) *
           (g->lon_edges[k + 1] - g->lon_edges[k]);
}

static int upper_index(const double *e, int n, double x)
{
    /* cell m with e[m] <= x < e[m+1], clamped to [0, n-1] */
    int m = 0;
    while (m < n - 1 && x >= e[m + 1]) ++m;
    return m;
}

static void locate(const geom_t *G, const double p[3], int ijk[3])
{
    double r = sqrt(dot3(p, p));
    ijk[0] = upper_index(G->R, G->nlev, r);
    double ct = r > 0 ? p[2] / r : 1.0;
    if (ct > 1.0) ct = 1.0;
    if (ct < -1.0) ct = -1.0;
    ijk[1] = G->nlat > 1 ? upper_index(G->th, G->nlat, acos(ct)) : 0;
    double phi = atan2(p[1], p[0]);
    if (phi < 0) phi += 2.0 * PI;
    ijk[2] = G->nlon > 1 ? upper_index(G->ph, G->nlon, phi) : 0;
}

void orc_locate(const orc_grid *g, const double p[3], int ijk[3])
{
    geom_t G;
    if (geom_init(&G, g)) return;
    locate(&G, p, ijk);
    geom_free(&G);
}

/* ------------------------------------------------------------------ */
/* O5: flight through the grid (algorithm C1).     */
/* ------------------------------------------------------------------ */
enum { ST_INTERACT = 0, ST_ESCAPE = 1, ST_SURFACE = 2, ST_STUCK = 3 };
enum { F_SHELL_OUT = 0, F_SHELL_IN, F_CONE_LO, F_CONE_HI, F_PLANE_LO, F_PLANE_HI };

static inline void take(double s, int face, double *smin, int *fmin)
{
    if (s < *smin) { *smin = s; *fmin = face; }   /* strict: ties keep the lower face id (C1) */
}

static void cone_candidates(const geom_t *G, int edge, int face, const double p[3], const double n[3],
                            double r2, double b, double *smin, int *fmin)
{
    double c = G->cth[edge];
    if (G->sth[edge] < 1e-12) return;               /* theta = 0 or pi: no surface (O5) */
    double z = p[2], nz = n[2];
    if (fabs(c) < 1e-12) {                           /* theta = pi/2: the plane z = 0 */
        if (nz != 0.0) {
            double s = -z / nz;
            if (s > G->s_eps) take(s, face, smin, fmin);
        }
        return;
    }
    double c2 = c * c;
    double A = nz * nz - c2;
    double B = z * nz - c2 * b;
    double C = z * z - c2 * r2;
    double s1, s2;
    int n_roots;
    if (fabs(A) < 1e-14) {
        if (B == 0.0) return;
        s1 = -C / (2.0 * B); s2 = s1; n_roots = 1;
    } else {
        double disc = B * B - A * C;
        if (disc < 0.0) return;
        double sq = sqrt(disc);
        double q = -(B + (B >= 0.0 ? sq : -sq));
        s1 = q / A;
        s2 = (q != 0.0) ? C / q : s1;
        n_roots = 2;
    }
    if (s1 > G->s_eps && (z + nz * s1) * c > 0.0) take(s1, face, smin, fmin);
    if (n_roots == 2 && s2 > G->s_eps && (z + nz * s2) * c > 0.0) take(s2, face, smin, fmin);
}

static void plane_candidate(const geom_t *G, int edge, int face, const double p[3], const double n[3],
                            double *smin, int *fmin)
{
    double cp = G->cph[edge], sp = G->sph[edge];
    double den = -n[0] * sp + n[1] * cp;             /* n . N, N = (-sin, cos, 0) */
    if (den == 0.0) return;
    double s = -(-p[0] * sp + p[1] * cp) / den;
    if (!(s > G->s_eps)) return;
    double hx = p[0] + n[0] * s, hy = p[1] + n[1] * s;
    if (hx * cp + hy * sp > 0.0) take(s, face, smin, fmin);   /* the half-plane, not its mirror */
}

/* Advance (p, ijk) along n until tau_limit is reached, the TOA is left, or the surface is hit. */
static int march2(const geom_t *G, const double *alpha, double p[3], const double n[3], int ijk[3],
                  double tau_limit, double *tau_out, uint64_t *nseg, double *path, const double *alpha_b, double *tau_b);
static int march(const geom_t *G, const double *alpha, double p[3], const double n[3], int ijk[3],
                 double tau_limit, double *tau_out, uint64_t *nseg, double *path)
{
    return march2(G, alpha, p, n, ijk, tau_limit, tau_out, nseg, path, NULL, NULL);
}
/* alpha_b (optional): a second extinction integrated over the same path into *tau_b (Eq. 12: tau_abs of the flight) */
static int march2(const geom_t *G, const double *alpha, double p[3], const double n[3], int ijk[3],
                  double tau_limit, double *tau_out, uint64_t *nseg, double *path, const double *alpha_b, double *tau_b)
{
    int i = ijk[0], j = ijk[1], k = ijk[2];
    double tau = 0.0;
    int status = ST_STUCK;
    for (int it = 0; it < G->maxseg; ++it) {
        double r2 = dot3(p, p), b = dot3(p, n);
        double smin = INFINITY;
        int face = -1;
        {   /* outer shell: always a candidate */
            double Ro = G->R[i + 1];
            double disc = b * b - (r2 - Ro * Ro);
            if (disc < 0.0) disc = 0.0;
            double s = -b + sqrt(disc);
            if (s < 0.0) s = 0.0;
            take(s, F_SHELL_OUT, &smin, &face);
        }
        if (b < 0.0) {   /* inner shell: only when moving inward and the ray reaches it */
            double Ri = G->R[i];
            double disc = b * b - (r2 - Ri * Ri);
            if (disc > 0.0) {
                double s = -b - sqrt(disc);
                if (s < 0.0) s = 0.0;
                take(s, F_SHELL_IN, &smin, &face);
            }
        }
        if (G->nlat > 1) {
            cone_candidates(G, j, F_CONE_LO, p, n, r2, b, &smin, &face);
            cone_candidates(G, j + 1, F_CONE_HI, p, n, r2, b, &smin, &face);
        }
        if (G->nlon > 1) {
            plane_candidate(G, k, F_PLANE_LO, p, n, &smin, &face);
            plane_candidate(G, k + 1, F_PLANE_HI, p, n, &smin, &face);
        }
        double a = alpha[cell_index(G, i, j, k)];
        ++*nseg;
        if (tau + a * smin >= tau_limit) {
            double s = (tau_limit - tau) / a;
            for (int m = 0; m < 3; ++m) p[m] += n[m] * s;
            if (path) *path += s;
            if (alpha_b) *tau_b += alpha_b[cell_index(G, i, j, k)] * s;
            tau = tau_limit;
            status = ST_INTERACT;
            break;
        }
        tau += a * smin;
        if (alpha_b) *tau_b += alpha_b[cell_index(G, i, j, k)] * smin;
        for (int m = 0; m < 3; ++m) p[m] += n[m] * smin;
        if (path) *path += smin;
        switch (face) {
        case F_SHELL_OUT: ++i; break;
        case F_SHELL_IN: --i; break;
        case F_CONE_LO: --j; break;
        case F_CONE_HI: ++j; break;
        case F_PLANE_LO: k = (k - 1 + G->nlon) % G->nlon; break;
        case F_PLANE_HI: k = (k + 1) % G->nlon; break;
        default: break;
        }
        if (i >= G->nlev) { i = G->nlev - 1; status = ST_ESCAPE; break; }
        if (i < 0) { i = 0; status = ST_SURFACE; break; }
        if (j < 0) j = 0;
        if (j >= G->nlat) j = G->nlat - 1;
    }
    ijk[0] = i; ijk[1] = j; ijk[2] = k;
    *tau_out = tau;
    return status;
}

/* ------------------------------------------------------------------ */
/* O9 / Eq. 33-34: Doppler shift.                                      */
/* ------------------------------------------------------------------ */
/* Eq. 33 exactly as printed, theta / theta_v colatitudes (C13). */
double orc_vlos_eq33(double u, double v, double w, double Omega, double r, double theta, double phi,
                     double theta_v, double phi_v)
{
    return u * sin(theta_v) * sin(phi - phi_v)
         + (v * cos(theta) - w * sin(theta)) * sin(theta_v) * cos(phi - phi_v)
         - (v * sin(theta) + w * cos(theta)) * cos(theta_v)
         + Omega * r * sin(theta) * sin(theta_v) * sin(phi - phi_v);
}
/* The same thing as -(u phi^ - v theta^ + w r^ + Omega r sin(theta) phi^) . o^  (C13). */
double orc_vlos_vector(double u, double v, double w, double Omega, double r, double theta, double phi,
                       const double obs[3])
{
    double st = sin(theta), ct = cos(theta), sp = sin(phi), cp = cos(phi);
    double phat[3] = { -sp, cp, 0.0 };
    double that[3] = { ct * cp, ct * sp, -st };
    double rhat[3] = { st * cp, st * sp, ct };
    double ue = u + Omega * r * st;
    double V[3];
    for (int m = 0; m < 3; ++m) V[m] = ue * phat[m] - v * that[m] + w * rhat[m];
    return -dot3(V, obs);
}

/* O9: kappa_abs of (channel c, cell) interpolated to lambda_eff = lambda_0 (1 - v_LOS/c) (Eq. 34),
 * linear in the wavelength index (C14), offset clamped to the +-W window and the table ends. */
static double doppler_kabs(const orc_grid *g, const orc_opacity *op, const geom_t *G, int W, int c, int i, int j, int k,
                           const double obs[3])
{
    int cell = cell_index(G, i, j, k);
    size_t nc = (size_t)G->ncell;
    if (op->n_chan < 2) return op->k_abs[(size_t)c * nc + cell];
    double rc = 0.5 * (G->R[i] + G->R[i + 1]);
    double thc = 0.5 * (G->th[j] + G->th[j + 1]);
    double phc = 0.5 * (G->ph[k] + G->ph[k + 1]);
    double uu = g->u ? g->u[cell] : 0.0, vv = g->v ? g->v[cell] : 0.0, ww = g->w ? g->w[cell] : 0.0;
    double vlos = orc_vlos_vector(uu, vv, ww, g->Omega, rc, thc, phc, obs);
    int c1 = (c + 1 < op->n_chan) ? c : c - 1;
    double Reff = 1.0 / log((double)op->lambda[c1 + 1] / (double)op->lambda[c1]);
    double dn = -vlos / C_LIGHT * Reff;
    if (dn > (double)W) dn = (double)W;
    if (dn < -(double)W) dn = -(double)W;
    double x = (double)c + dn;
    if (x < 0.0) x = 0.0;
    if (x > (double)(op->n_chan - 1)) x = (double)(op->n_chan - 1);
    int lo = (int)floor(x);
    if (lo > op->n_chan - 2) lo = op->n_chan - 2;
    double f = x - (double)lo;
    double k0 = op->k_abs[(size_t)lo * nc + cell], k1 = op->k_abs[(size_t)(lo + 1) * nc + cell];
    return (1.0 - f) * k0 + f * k1;
}

/* ------------------------------------------------------------------ */
/* O2: channel preparation (A0, A1, A2).                               */
/* ------------------------------------------------------------------ */
typedef struct {
    double *alpha, *omega, *pgas, *gg, *Lcum; /* [ncell] each; Lcum = running sum of L_i */
    double *Lcell;
    double *alpha_sca, *alpha_abs;            /* rho kappa_sca, rho kappa_abs (continuous absorption, Eq. 12) */
    double L_tot;
} chan_t;

static int chan_alloc(chan_t *ch, int ncell)
{
    ch->alpha = (double *)malloc(sizeof(double) * (size_t)ncell * 8);
    if (!ch->alpha) return -1;
    ch->omega = ch->alpha + ncell; ch->pgas = ch->omega + ncell; ch->gg = ch->pgas + ncell;
    ch->Lcell = ch->gg + ncell; ch->Lcum = ch->Lcell + ncell;
    ch->alpha_sca = ch->Lcum + ncell; ch->alpha_abs = ch->alpha_sca + ncell;
    ch->L_tot = 0.0;
    return 0;
}
static void chan_free(chan_t *ch) { free(ch->alpha); }

static void chan_prep(const orc_grid *g, const geom_t *G, const orc_opacity *op, const orc_params *prm, int c,
                      int obs_index, int emission, chan_t *ch)
{
    size_t nc = (size_t)G->ncell;
    const double *obs = (prm->doppler_on && obs_index >= 0) ? prm->obs_dir + 3 * obs_index : NULL;
    for (int k = 0; k < G->nlon; ++k)
        for (int j = 0; j < G->nlat; ++j)
            for (int i = 0; i < G->nlev; ++i) {
                int cell = cell_index(G, i, j, k);
                double rho = g->rho[cell];
                double ka = obs ? doppler_kabs(g, op, G, prm->doppler_halfwidth, c, i, j, k, obs)
                                : (double)op->k_abs[(size_t)c * nc + cell];
                double kr = op->k_sca_ray ? op->k_sca_ray[(size_t)c * nc + cell] : 0.0;
                double kc = op->k_sca_cld ? op->k_sca_cld[(size_t)c * nc + cell] : 0.0;
                double ks = kr + kc;
                double kext = ka + ks;
                ch->alpha[cell] = rho * kext;                       /* alpha_ext */
                ch->alpha_sca[cell] = rho * ks;
                ch->alpha_abs[cell] = rho * ka;
                ch->omega[cell] = kext > 0.0 ? ks / kext : 0.0;     /* single-scattering albedo */
                ch->pgas[cell] = ks > 0.0 ? kr / ks : 0.0;          /* Eq. 11 */
                ch->gg[cell] = op->g_cld ? op->g_cld[(size_t)c * nc + cell] : 0.0;
                ch->Lcell[cell] = 0.0;
                if (emission) {
                    /* Eq. 27: L_i = 4 pi V_i rho_i kappa_abs,i B_lambda(T_i) */
                    ch->Lcell[cell] = 4.0 * PI * orc_cell_volume(g, i, j, k) * rho * ka *
                                      orc_planck((double)op->lambda[c], (double)g->T[cell]);
                }
            }
    ch->L_tot = 0.0;
    if (emission) {
        /* L210 / C15: drop cells whose vertical optical depth from the TOA to their upper face exceeds tau_vert_max */
        if (prm->tau_vert_max > 0.0) {
            for (int k = 0; k < G->nlon; ++k)
                for (int j = 0; j < G->nlat; ++j) {
                    double tv = 0.0;
                    for (int i = G->nlev - 1; i >= 0; --i) {
                        int cell = cell_index(G, i, j, k);
                        if (tv > prm->tau_vert_max) ch->Lcell[cell] = 0.0;
                        tv += ch->alpha[cell] * (G->R[i + 1] - G->R[i]);
                    }
                }
        }
        double run = 0.0;
        for (int cell = 0; cell < G->ncell; ++cell) { run += ch->Lcell[cell]; ch->Lcum[cell] = run; }
        ch->L_tot = run;
    }
}

int orc_channel_prep(const orc_grid *g, const orc_opacity *op, const orc_params *prm, int chan, int obs_index,
                     double *alpha, double *omega, double *pgas, double *gg, double *L_cell, double *L_tot)
{
    geom_t G;
    chan_t ch;
    if (geom_init(&G, g)) return -1;
    if (chan_alloc(&ch, G.ncell)) { geom_free(&G); return -1; }
    chan_prep(g, &G, op, prm, chan, obs_index, L_cell != NULL, &ch);
    size_t nb = sizeof(double) * (size_t)G.ncell;
    if (alpha) memcpy(alpha, ch.alpha, nb);
    if (omega) memcpy(omega, ch.omega, nb);
    if (pgas) memcpy(pgas, ch.pgas, nb);
    if (gg) memcpy(gg, ch.gg, nb);
    if (L_cell) memcpy(L_cell, ch.Lcell, nb);
    if (L_tot) *L_tot = ch.L_tot;
    chan_free(&ch);
    geom_free(&G);
    return 0;
}

int orc_ray_tau(const orc_grid *g, const orc_opacity *op, int chan, long n, const double *pos, const double *dir,
                double *tau, int *hit_surface, long *nseg_out, double *path_len)
{
    geom_t G;
    chan_t ch;
    orc_params prm;
    memset(&prm, 0, sizeof prm);
    if (geom_init(&G, g)) return -1;
    if (chan_alloc(&ch, G.ncell)) { geom_free(&G); return -1; }
    chan_prep(g, &G, op, &prm, chan, -1, 0, &ch);
    for (long m = 0; m < n; ++m) {
        double p[3] = { pos[3 * m], pos[3 * m + 1], pos[3 * m + 2] };
        double d[3] = { dir[3 * m], dir[3 * m + 1], dir[3 * m + 2] };
        int ijk[3];
        locate(&G, p, ijk);
        uint64_t nseg = 0;
        double path = 0.0, t = 0.0;
        int st = march(&G, ch.alpha, p, d, ijk, INFINITY, &t, &nseg, &path);
        tau[m] = t;
        if (hit_surface) hit_surface[m] = (st == ST_SURFACE) ? 1 : (st == ST_STUCK ? -1 : 0);
        if (nseg_out) nseg_out[m] = (long)nseg;
        if (path_len) path_len[m] = path;
    }
    chan_free(&ch);
    geom_free(&G);
    return 0;
}

/* ------------------------------------------------------------------ */
/* O3..O8: packets.                                                    */
/* ------------------------------------------------------------------ */
typedef struct {
    const orc_grid *g;
    const geom_t *G;
    const orc_params *prm;
    const chan_t *ch;
    int c;             /* local channel */
    uint32_t chan_key; /* global channel = Philox key[0] */
    int obs_lo, obs_hi; /* observers peeled in this run */
    double e1[3], e2[3]; /* launch disc basis (O3) */
    double *S;         /* flux_sum for this channel: [n_obs][n_batches] */
    double *image;     /* this channel's [n_obs][npix][npix] or NULL */
    double *contrib;   /* this channel's [n_obs][2][ncell] or NULL (Sect. 6, Eq. 32) */
    uint32_t *evcount; /* this channel's [N] or NULL */
    int launch_forced; /* packet_albedo -> transport: the launch flight was forced (and stretched there) */
    double peel_scale; /* what a peeled-off f adds to S: 1 (albedo, emission); -W_ld b dOmega for the scattered light of a
                          transit chord (Sect. 5.1 with multiple scattering, reading N12) */
} run_ctx;

/* C19: image pixel of point p seen from observer direction o. */
static int image_pixel(const double p[3], const double o[3], double Rtoa, int npix)
{
    double ex[3] = { -o[1], o[0], 0.0 };   /* z^ x o^ */
    double nn = sqrt(ex[0] * ex[0] + ex[1] * ex[1]);
    if (nn < 1e-6) { ex[0] = 1.0; ex[1] = 0.0; ex[2] = 0.0; } else { ex[0] /= nn; ex[1] /= nn; }
    double ey[3] = { o[1] * ex[2] - o[2] * ex[1], o[2] * ex[0] - o[0] * ex[2], o[0] * ex[1] - o[1] * ex[0] };
    double X = dot3(p, ex), Y = dot3(p, ey);
    int ix = (int)floor((X / Rtoa + 1.0) * 0.5 * npix);
    int iy = (int)floor((Y / Rtoa + 1.0) * 0.5 * npix);
    if (ix < 0) ix = 0;
    if (ix >= npix) ix = npix - 1;
    if (iy < 0) iy = 0;
    if (iy >= npix) iy = npix - 1;
    return iy * npix + ix;
}

/* Eq. 14: peel the fraction `pref * exp(-tau_obs)` to every observer of this run.
 * pref_of(o) is W*omega*Theta (medium), W/(4pi) (emission) or W*a*max(n^.o,0)/pi (surface). */
static void peel(const run_ctx *rc, const double p[3], const int ijk[3], int kind, double W, const double nin[3],
                 double omega, double pgas, double gg, int batch, orc_counters *cnt)
{
    const geom_t *G = rc->G;
    for (int o = rc->obs_lo; o < rc->obs_hi; ++o) {
        const double *od = rc->prm->obs_dir + 3 * o;
        double pref;
        if (kind == 0) {            /* medium interaction, C6: mixture phase function */
            double mu = dot3(nin, od);
            double cld = rc->prm->cloud_phase == 1 ? orc_phase_tthg(gg, mu)
                       : rc->prm->cloud_phase == 2 ? orc_phase_draine(gg, mu) : orc_phase_hg(gg, mu);
            double theta = pgas * orc_phase_rayleigh(mu) + (1.0 - pgas) * cld;
            pref = W * omega * theta;
        } else if (kind == 1) {     /* thermal emission: isotropic, no omega (O4) */
            pref = W / (4.0 * PI);
        } else {                    /* Lambert surface (O7): nin holds the surface normal */
            double mu = dot3(nin, od);
            if (mu <= 0.0) continue;
            pref = W * omega * mu / PI;   /* omega carries the surface albedo here */
        }
        double q[3] = { p[0], p[1], p[2] };
        int c3[3] = { ijk[0], ijk[1], ijk[2] };
        double tau = 0.0;
        int st = march(G, rc->ch->alpha, q, od, c3, INFINITY, &tau, &cnt->segments_peel, NULL);
        if (st != ST_ESCAPE) continue;                 /* ray ends on the surface: nothing reaches the observer */
        if (tau > rc->prm->tau_cut) continue;
        double f = rc->peel_scale * pref * exp(-tau);
        rc->S[(size_t)o * rc->prm->n_batches + batch] += f;
        if (rc->image) {
            int npix = rc->prm->npix;
            rc->image[(size_t)o * npix * npix + image_pixel(p, od, G->Rtoa, npix)] += f;
        }
        if (rc->contrib)   /* Sect. 6: the contribution of the event's cell to the output, thermal / scattered apart */
            rc->contrib[((size_t)o * 2 + (kind == 1 ? 0 : 1)) * G->ncell + cell_index(G, ijk[0], ijk[1], ijk[2])] += f;
    }
}

/* Cloud scatterer: HG, or TTHG whose lobe is picked by the part of zeta0 left over inside the cloud interval of the
 * partition (uniform in [0,1) given that the cloud was chosen), so that no extra draw is needed. */
static double sample_cloud(const orc_params *prm, double gg, double zlobe, double zeta)
{
    if (prm->cloud_phase == 2) return orc_sample_draine(gg, zeta);
    return prm->cloud_phase == 1 ? orc_sample_tthg(gg, zlobe, zeta) : orc_sample_hg(gg, zeta);
}

/* O6/O7/O5 loop shared by both modes.  m = number of peel-off points so far. */
static void transport(const run_ctx *rc, uint32_t pkt, double p[3], double n[3], int ijk[3], double W, double tau_t,
                      uint32_t m, int batch, orc_counters *cnt)
{
    const geom_t *G = rc->G;
    const orc_params *prm = rc->prm;
    const chan_t *ch = rc->ch;
    const double a_surf = rc->g->surface_albedo;
    uint32_t m_inter = 0;    /* interaction index (Philox event index), 1,2,... */
    double z[4];
    const int cont = prm->continuous_absorption != 0;
    /* Sect. 4.2, path length stretching (Baes et al. 2016): flights are drawn from the stretched law
     * q(tau) = a e^{-a tau} (a = stretch_alpha < 1: longer flights) instead of p(tau) = e^{-tau}, and the packet carries
     * the ratio p / q of what happened to it: an interaction at tau, W <- W e^{-(1-a) tau} / a; leaving the medium
     * (top or lower boundary) after tau_edge, W <- W e^{-(1-a) tau_edge} (the ratio of the two survival probabilities).
     * Hybrid with forced scattering: the stretched law truncated at tau_edge, q = a e^{-a tau} / (1 - e^{-a tau_edge}),
     * so the interaction weight gains the factor 1 - e^{-a tau_edge} and the uncollided part W e^{-tau_edge} leaves. */
    const double sa = (prm->stretch_alpha > 0.0 && prm->stretch_alpha < 1.0) ? prm->stretch_alpha : 1.0;
    int flight = 0;
    for (;;) {
        double tau = 0.0;
        int st;
        const int launch_flight = (flight++ == 0 && m == 0);   /* the flight packet_albedo prepared (m == 0: albedo) */
        int forced_now = launch_flight ? rc->launch_forced : 0;   /* ... and forced (and stretched) there */
        if (prm->forced_scatter == 2 && !launch_flight) {
            /* Sect. 4.2, forced scattering at every flight (the albedo launch does it for the first one): the flight is
             * drawn from the exponential law truncated at the optical depth to the end of the grid, the packet keeps
             * the probability 1 - e^-tau_edge of interacting, the uncollided part leaves (Cashwell & Everett 1959) */
            double q[3] = { p[0], p[1], p[2] }, tau_edge = 0.0;
            int c3[3] = { ijk[0], ijk[1], ijk[2] };
            uint64_t seg = 0;
            int se = march(G, ch->alpha, q, n, c3, INFINITY, &tau_edge, &seg, NULL);
            if (se == ST_ESCAPE || (se == ST_SURFACE && !(a_surf > 0.0))) {
                const double pint = -expm1(-sa * tau_edge);     /* sa = 1: the plain forced flight */
                if (pint > 0.0) {
                    if (se == ST_ESCAPE) cnt->escaped_weight += W * exp(-tau_edge);
                    tau_t = -log1p(-exp(-tau_t) * pint) / sa;   /* the flight's own zeta = e^-tau_t */
                    W *= pint;
                    forced_now = 1;
                }
            }
        }
        if (sa < 1.0 && !forced_now) tau_t /= sa;               /* tau = -ln(zeta) / a */
        if (cont) {
            /* Sect. 4.1, Eq. 12: the sampled optical depth is spent on the scattering extinction alone and the packet
             * loses weight smoothly, W <- W e^-tau_abs, with tau_abs integrated along the same flight */
            double tau_abs = 0.0;
            st = march2(G, ch->alpha_sca, p, n, ijk, tau_t, &tau, &cnt->segments_transport, NULL, ch->alpha_abs, &tau_abs);
            W *= exp(-tau_abs);
        } else {
            st = march(G, ch->alpha, p, n, ijk, tau_t, &tau, &cnt->segments_transport, NULL);
        }
        if (sa < 1.0) {   /* p / q of the flight's outcome */
            if (st == ST_INTERACT) W *= exp(-(1.0 - sa) * tau_t) / sa;
            else if (st == ST_ESCAPE || st == ST_SURFACE) W *= exp(-(1.0 - sa) * tau);
        }
        if (st == ST_ESCAPE) { cnt->packets_escaped++; cnt->escaped_weight += W; break; }
        if (st == ST_STUCK) { cnt->packets_stuck++; break; }
        if (st == ST_SURFACE) {
            if (!(a_surf > 0.0)) { cnt->packets_surface++; break; }
            /* O7: Lambert surface, Eq. 3-4 */
            ++m_inter; ++m; cnt->events++;
            orc_zeta_block(prm->seed, rc->chan_key, pkt, m_inter, 3, z);
            double rr = sqrt(dot3(p, p));
            double nh[3] = { p[0] / rr, p[1] / rr, p[2] / rr };
            peel(rc, p, ijk, 2, W, nh, a_surf, 0.0, 0.0, batch, cnt);
            if (prm->max_events && (int)m_inter == prm->max_events) { cnt->packets_absorbed++; break; }
            if (z[0] >= a_surf) { cnt->packets_surface++; break; }
            orc_rotate(nh, orc_sample_lambert(z[1]), 2.0 * PI * z[2], n);
            tau_t = -log(z[3]);
            continue;
        }
        /* O6: interaction in the medium */
        ++m_inter; ++m; cnt->events++;
        orc_zeta_block(prm->seed, rc->chan_key, pkt, m_inter, 1, z);
        int cell = cell_index(G, ijk[0], ijk[1], ijk[2]);
        double omega = ch->omega[cell], pgas = ch->pgas[cell], gg = ch->gg[cell];
        if (cont) omega = 1.0;   /* the interaction was drawn from the scattering extinction: it is a scattering (Eq. 14
                                    without the albedo factor; the absorbed part already left the weight, Eq. 12) */
        peel(rc, p, ijk, 0, W, n, omega, pgas, gg, batch, cnt);     /* peel-off first (Sect. 4.6) */
        if (prm->max_events && (int)m_inter == prm->max_events) { cnt->packets_absorbed++; break; }
        if (!prm->scatter_on) { cnt->packets_absorbed++; break; }
        double ct;
        if (prm->survival_bias) {
            /* Sect. 4.4: the packet is forced to scatter and its weight reduced by omega; the draw that
             * decides absorption in the analog scheme only picks the scatterer (Eq. 11: gas with probability P_gas) */
            if (!(omega > 0.0)) { cnt->packets_absorbed++; break; }
            W *= omega;
            /* Sect. 4.5: Russian roulette below the weight threshold; block (m_inter, purpose 2) */
            if (prm->roulette_w_min > 0.0 && W < prm->roulette_w_min) {
                double zr[4];
                orc_zeta_block(prm->seed, rc->chan_key, pkt, m_inter, 2, zr);
                if (zr[0] >= prm->roulette_survive) { cnt->packets_absorbed++; break; }
                W /= prm->roulette_survive;
            }
            ct = (z[0] < pgas) ? orc_sample_rayleigh(z[1]) : sample_cloud(prm, gg, (z[0] - pgas) / (1.0 - pgas), z[1]);
        } else {
            if (z[0] >= omega) { cnt->packets_absorbed++; break; }     /* Sect. 4.4: analog absorption */
            ct = (z[0] < omega * pgas) ? orc_sample_rayleigh(z[1])  /* Eq. 11 + C6 partition */
                                       : sample_cloud(prm, gg, (z[0] - omega * pgas) / (omega - omega * pgas), z[1]);
        }
        double nn[3];
        orc_rotate(n, ct, 2.0 * PI * z[2], nn);
        n[0] = nn[0]; n[1] = nn[1]; n[2] = nn[2];
        tau_t = -log(z[3]);
    }
    if (rc->evcount) rc->evcount[pkt] = m;
}

/* Sect. 4.2: "an extra raytracing step to calculate the optical depth to the end of the grid in the direction of
 * the packet path", at the start of a packet (forced first scattering; with forced_scatter = 2 the later flights are
 * forced in transport()).  The flight is drawn from the exponential law truncated at tau_edge and the packet carries the
 * probability 1 - e^-tau_edge that an analog packet interacts at all (Cashwell & Everett 1959); with path length
 * stretching (sa < 1) the stretched law is truncated instead (the hybrid scheme).  Returns 1 when the flight was forced,
 * 0 when not (forcing off, or the ray ends on a reflecting lower boundary), -1 when the path is empty (the packet ends). */
static int forced_launch(const run_ctx *rc, const double p[3], const double n[3], const int ijk[3], double zeta,
                         double *W, double *tau_t, orc_counters *cnt)
{
    const orc_params *prm = rc->prm;
    if (!prm->forced_scatter) return 0;
    const double sa = (prm->stretch_alpha > 0.0 && prm->stretch_alpha < 1.0) ? prm->stretch_alpha : 1.0;
    double q[3] = { p[0], p[1], p[2] }, tau_edge = 0.0;
    int c3[3] = { ijk[0], ijk[1], ijk[2] };
    uint64_t seg = 0;
    int st = march(rc->G, rc->ch->alpha, q, n, c3, INFINITY, &tau_edge, &seg, NULL);
    if (!(st == ST_ESCAPE || (st == ST_SURFACE && !(rc->g->surface_albedo > 0.0)))) return 0;
    const double pint = -expm1(-sa * tau_edge);
    if (!(pint > 0.0)) {            /* empty path: nothing can interact, the packet ends with no event */
        if (st == ST_ESCAPE) { cnt->packets_escaped++; cnt->escaped_weight += *W; } else cnt->packets_surface++;
        return -1;
    }
    if (st == ST_ESCAPE) cnt->escaped_weight += *W * exp(-tau_edge);   /* the part that leaves without interacting */
    *W *= pint;
    *tau_t = -log1p(-zeta * pint) / sa;
    return 1;
}

/* O3: albedo launch. */
static void packet_albedo(const run_ctx *rc, uint32_t pkt, int batch, orc_counters *cnt)
{
    const geom_t *G = rc->G;
    const orc_params *prm = rc->prm;
    double z[4];
    orc_zeta_block(prm->seed, rc->chan_key, pkt, 0, 0, z);
    double b = G->Rtoa * sqrt(z[0]);
    double psi = 2.0 * PI * z[1];
    double h = sqrt(fmax(0.0, G->Rtoa * G->Rtoa - b * b));
    double p[3], n[3];
    for (int m = 0; m < 3; ++m) {
        p[m] = b * cos(psi) * rc->e1[m] + b * sin(psi) * rc->e2[m] + h * prm->star_dir[m];
        n[m] = -prm->star_dir[m];
    }
    int ijk[3];
    locate(G, p, ijk);
    ijk[0] = G->nlev - 1;
    double W = 1.0, tau_t = -log(z[2]);
    run_ctx rcl = *rc;
    rcl.launch_forced = forced_launch(rc, p, n, ijk, z[2], &W, &tau_t, cnt);
    if (rcl.launch_forced < 0) { if (rc->evcount) rc->evcount[pkt] = 0; return; }
    transport(&rcl, pkt, p, n, ijk, W, tau_t, 0, batch, cnt);
}

/* O4: emission launch (Eq. 13, Sect. 4.3 with the C10 composite bias). */
static void packet_emission(const run_ctx *rc, uint32_t pkt, int batch, orc_counters *cnt)
{
    const geom_t *G = rc->G;
    const orc_params *prm = rc->prm;
    const chan_t *ch = rc->ch;
    double z[4];
    orc_zeta_block(prm->seed, rc->chan_key, pkt, 0, 0, z);
    double xi = prm->emission_bias;
    int cell;
    if (z[0] < xi) {
        cell = (int)floor(z[0] / xi * G->ncell);
        if (cell >= G->ncell) cell = G->ncell - 1;
    } else {
        double x = (z[0] - xi) / (1.0 - xi) * ch->L_tot;
        /* first cell whose running luminosity exceeds x */
        int lo = 0, hi = G->ncell - 1;
        while (lo < hi) {
            int mid = (lo + hi) / 2;
            if (ch->Lcum[mid] > x) hi = mid; else lo = mid + 1;
        }
        cell = lo;
    }
    double Li = ch->Lcell[cell];
    if (!(Li > 0.0)) { if (rc->evcount) rc->evcount[pkt] = 0; return; }   /* zero-luminosity cell: W = 0 */
    double W = 1.0 / ((1.0 - xi) + xi * ch->L_tot / ((double)G->ncell * Li));
    int i = cell % G->nlev, j = (cell / G->nlev) % G->nlat, k = cell / (G->nlev * G->nlat);
    double R0 = G->R[i], R1 = G->R[i + 1];
    double r = cbrt(R0 * R0 * R0 + z[1] * (R1 * R1 * R1 - R0 * R0 * R0));
    double ct = G->cth[j] + z[2] * (G->cth[j + 1] - G->cth[j]);
    double st = sqrt(fmax(0.0, 1.0 - ct * ct));
    double phi = G->ph[k] + z[3] * (G->ph[k + 1] - G->ph[k]);
    double p[3] = { r * st * cos(phi), r * st * sin(phi), r * ct };
    orc_zeta_block(prm->seed, rc->chan_key, pkt, 1, 0, z);
    double nz = orc_sample_isotropic(z[0]);                       /* Eq. 2 */
    double ns = sqrt(fmax(0.0, 1.0 - nz * nz));
    double psi = 2.0 * PI * z[1];
    double n[3] = { ns * cos(psi), ns * sin(psi), nz };
    int ijk[3] = { i, j, k };
    cnt->events++;
    peel(rc, p, ijk, 1, W, n, 0.0, 0.0, 0.0, batch, cnt);         /* initial peel-off (L210) */
    if (!prm->scatter_on) { cnt->packets_absorbed++; if (rc->evcount) rc->evcount[pkt] = 1; return; }
    transport(rc, pkt, p, n, ijk, W, -log(z[2]), 1, batch, cnt);
}

static void add_counters(orc_counters *a, const orc_counters *b)
{
    a->events += b->events;
    a->segments_transport += b->segments_transport;
    a->segments_peel += b->segments_peel;
    a->packets_escaped += b->packets_escaped;
    a->packets_absorbed += b->packets_absorbed;
    a->packets_surface += b->packets_surface;
    a->packets_stuck += b->packets_stuck;
    a->escaped_weight += b->escaped_weight;
}

static int run_mode(const orc_grid *g, const orc_opacity *op, const orc_params *prm, orc_result *out, int emission)
{
    geom_t G;
    if (!g || !op || !prm || !out || prm->n_batches < 1 || prm->n_obs < 0) return -1;
    if (geom_init(&G, g)) return -1;
    const uint64_t N = prm->packets_per_channel;
    const int nb = prm->n_batches, nobs = prm->n_obs;
    const int npix = prm->npix;
    memset(&out->counters, 0, sizeof out->counters);
    memset(out->flux_sum, 0, sizeof(double) * (size_t)op->n_chan * nobs * nb);
    if (out->image && npix > 0) memset(out->image, 0, sizeof(double) * (size_t)op->n_chan * nobs * npix * npix);
    if (out->contrib) memset(out->contrib, 0, sizeof(double) * (size_t)op->n_chan * nobs * 2 * G.ncell);
    int nthreads = prm->n_threads > 1 ? prm->n_threads : 1;
    chan_t ch;
    if (chan_alloc(&ch, G.ncell)) { geom_free(&G); return -1; }

    /* with doppler_on every observer is an independent run with its own shifted table (L326-328, O9) */
    int n_runs = prm->doppler_on ? nobs : 1;
    for (int c = 0; c < op->n_chan; ++c) {
        for (int run = 0; run < n_runs; ++run) {
            int obs_index = prm->doppler_on ? run : -1;
            chan_prep(g, &G, op, prm, c, obs_index, emission, &ch);
            if (out->L_tot) {
                if (prm->doppler_on) out->L_tot[(size_t)c * nobs + run] = ch.L_tot;
                else for (int o = 0; o < nobs; ++o) out->L_tot[(size_t)c * nobs + o] = ch.L_tot;
            }
            run_ctx rc;
            rc.g = g; rc.G = &G; rc.prm = prm; rc.ch = &ch; rc.c = c;
            rc.chan_key = (uint32_t)(op->chan0 + c);
            rc.obs_lo = prm->doppler_on ? run : 0;
            rc.obs_hi = prm->doppler_on ? run + 1 : nobs;
            {   /* O3: e1 = normalize(z^ x s^) (x^ if degenerate), e2 = s^ x e1 */
                const double *s = prm->star_dir;
                double e1[3] = { -s[1], s[0], 0.0 };
                double nn = sqrt(e1[0] * e1[0] + e1[1] * e1[1]);
                if (nn < 1e-6) { e1[0] = 1.0; e1[1] = 0.0; e1[2] = 0.0; } else { e1[0] /= nn; e1[1] /= nn; }
                rc.e1[0] = e1[0]; rc.e1[1] = e1[1]; rc.e1[2] = e1[2];
                rc.e2[0] = s[1] * e1[2] - s[2] * e1[1];
                rc.e2[1] = s[2] * e1[0] - s[0] * e1[2];
                rc.e2[2] = s[0] * e1[1] - s[1] * e1[0];
            }
            rc.S = out->flux_sum + (size_t)c * nobs * nb;
            rc.image = (out->image && npix > 0) ? out->image + (size_t)c * nobs * npix * npix : NULL;
            rc.contrib = out->contrib ? out->contrib + (size_t)c * nobs * 2 * G.ncell : NULL;
            rc.evcount = (out->event_count && run == 0) ? out->event_count + (size_t)c * N : NULL;
            rc.launch_forced = 0;
            rc.peel_scale = 1.0;
            if (emission && !(ch.L_tot > 0.0)) continue;
            /* O8 / C12: batch(pkt) = floor(pkt * n_batches / N); batches are independent -> OpenMP over them */
#ifdef _OPENMP
#pragma omp parallel for schedule(dynamic, 1) num_threads(nthreads) if (nthreads > 1 && !rc.image && !rc.contrib)
#endif
            for (int b = 0; b < nb; ++b) {
                orc_counters cnt;
                memset(&cnt, 0, sizeof cnt);
                /* packets of batch b: ceil(b N / nb) .. ceil((b+1) N / nb) - 1 */
                uint64_t lo = ((uint64_t)b * N + nb - 1) / nb, hi = ((uint64_t)(b + 1) * N + nb - 1) / nb;
                if (lo < prm->pkt_begin) lo = prm->pkt_begin;
                if (hi > prm->pkt_end) hi = prm->pkt_end;
                for (uint64_t pkt = lo; pkt < hi; ++pkt) {
                    if (emission) packet_emission(&rc, (uint32_t)pkt, b, &cnt);
                    else packet_albedo(&rc, (uint32_t)pkt, b, &cnt);
                }
#ifdef _OPENMP
#pragma omp critical
#endif
                add_counters(&out->counters, &cnt);
            }
        }
    }
    (void)nthreads;
    chan_free(&ch);
    geom_free(&G);
    return 0;
}

int orc_run_albedo(const orc_grid *g, const orc_opacity *op, const orc_params *prm, orc_result *out)
{
    return run_mode(g, op, prm, out, 0);
}

int orc_run_emission(const orc_grid *g, const orc_opacity *op, const orc_params *prm, orc_result *out)
{
    return run_mode(g, op, prm, out, 1);
}

/* ---- Sect. 5.1: transmission by random transit chords (Eq. 20-23) ------------------------------------------------
 * Packet pkt of channel c, Philox block (event 0, purpose 0): b = R_p0 + zeta0 (R_TOA - R_p0) (uniform in b: Eq. 21
 * carries the factor b_i explicitly), psi = 2 pi zeta1 around the limb.  The chord runs along o^ (planet -> observer)
 * through the point b (cos psi e_x + sin psi e_y) of the sky plane; it starts on the star side of the TOA sphere.
 * tau_i = extinction optical depth of the whole chord (the "initial peeloff", L255).  Chords never meet the lower
 * boundary because b >= R_p0 (L257).  Limb darkening: the chord's sky position relative to the stellar disc centre
 * gives mu = sqrt(1 - rho^2 / R_star^2) and W = 1 - c1 (1 - mu) - c2 (1 - mu)^2 (Eq. 22-23); off the disc W = 0. */
int orc_run_transmission(const orc_grid *g, const orc_opacity *op, const orc_params *prm, orc_result *out)
{
    geom_t G;
    if (!g || !op || !prm || !out || prm->n_batches < 1 || prm->n_obs < 1) return -1;
    if (geom_init(&G, g)) return -1;
    const uint64_t N = prm->packets_per_channel;
    const int nb = prm->n_batches, nobs = prm->n_obs;
    memset(&out->counters, 0, sizeof out->counters);
    memset(out->flux_sum, 0, sizeof(double) * (size_t)op->n_chan * nobs * nb);
    chan_t ch;
    if (chan_alloc(&ch, G.ncell)) { geom_free(&G); return -1; }
    const double R0 = G.R[0], Rt = G.Rtoa;
    for (int c = 0; c < op->n_chan; ++c) {
        for (int o = 0; o < nobs; ++o) {
            /* with doppler_on the observer's shifted table (O9); the unshifted one otherwise */
            if (o == 0 || prm->doppler_on) chan_prep(g, &G, op, prm, c, prm->doppler_on ? o : -1, 0, &ch);
            const double *od = prm->obs_dir + 3 * o;
            double ex[3] = { -od[1], od[0], 0.0 };   /* C19 frame */
            double nn = sqrt(ex[0] * ex[0] + ex[1] * ex[1]);
            if (nn < 1e-6) { ex[0] = 1.0; ex[1] = 0.0; ex[2] = 0.0; } else { ex[0] /= nn; ex[1] /= nn; }
            double ey[3] = { od[1] * ex[2] - od[2] * ex[1], od[2] * ex[0] - od[0] * ex[2], od[0] * ex[1] - od[1] * ex[0] };
            for (uint64_t pkt = prm->pkt_begin; pkt < prm->pkt_end; ++pkt) {
                double z[4];
                orc_zeta_block(prm->seed, (uint32_t)(op->chan0 + c), (uint32_t)pkt, 0, 0, z);
                const double b = R0 + z[0] * (Rt - R0), psi = 2.0 * PI * z[1];
                const double X = b * cos(psi), Y = b * sin(psi), h = sqrt(fmax(0.0, Rt * Rt - b * b));
                double p[3], q[3];
                for (int m = 0; m < 3; ++m) { p[m] = X * ex[m] + Y * ey[m] - h * od[m]; q[m] = p[m]; }
                double W = 1.0;
                if (prm->star_radius > 0.0) {
                    const double sx = prm->planet_xy[0] + X, sy = prm->planet_xy[1] + Y;
                    const double rho2 = (sx * sx + sy * sy) / (prm->star_radius * prm->star_radius);
                    if (rho2 >= 1.0) W = 0.0;
                    else { const double mu = sqrt(1.0 - rho2); W = 1.0 - prm->ld_c1 * (1.0 - mu) - prm->ld_c2 * (1.0 - mu) * (1.0 - mu); }
                }
                int ijk[3];
                locate(&G, q, ijk);
                ijk[0] = G.nlev - 1;
                double tau = 0.0;
                int st = march(&G, ch.alpha, q, od, ijk, INFINITY, &tau, &out->counters.segments_peel, NULL);
                out->counters.events++;
                if (st == ST_STUCK) { out->counters.packets_stuck++; continue; }
                const double absorbed = (st == ST_SURFACE) ? 1.0 : 1.0 - exp(-tau);   /* (a chord grazing R_p0 in fp) */
                const int batch = (int)((pkt * (uint64_t)nb) / N);
                out->flux_sum[((size_t)c * nobs + o) * nb + batch] += W * absorbed * b;
                if (prm->scatter_on && prm->star_solid_angle > 0.0 && W > 0.0) {
                    /* Sect. 5.1, L259 (reading N12): after the initial peel-off above "the packet is then free to multiply
                     * scatter through the atmosphere, each time contributing to the transmission ... through the next
                     * event estimation method".  The packet flies from the chord's start along o^ (tau = -ln zeta2 of
                     * the launch block); every interaction peels W omega Theta e^{-tau_obs} toward o^ (per steradian), and
                     * the observer receives that light as starlight over the solid angle of the stellar disc,
                     * star_solid_angle: the chord's term of Eq. 21 becomes
                     * W_ph b [1 - e^{-tau_i} - dOmega sum_k W_k omega_k Theta_k e^{-tau_obs,k}]. */
                    run_ctx rc;
                    memset(&rc, 0, sizeof rc);
                    rc.g = g; rc.G = &G; rc.prm = prm; rc.ch = &ch; rc.c = c;
                    rc.chan_key = (uint32_t)(op->chan0 + c);
                    rc.obs_lo = o; rc.obs_hi = o + 1;
                    rc.S = out->flux_sum + (size_t)c * nobs * nb;
                    rc.evcount = (out->event_count && o == 0) ? out->event_count + (size_t)c * N : NULL;
                    rc.launch_forced = 0;
                    rc.peel_scale = -W * b * prm->star_solid_angle;
                    double pp[3] = { p[0], p[1], p[2] }, nn3[3] = { od[0], od[1], od[2] };
                    int c3[3];
                    locate(&G, pp, c3);
                    c3[0] = G.nlev - 1;
                    orc_counters cnt;
                    memset(&cnt, 0, sizeof cnt);
                    double Wp = 1.0, tau_t = -log(z[2]);
                    rc.launch_forced = forced_launch(&rc, pp, nn3, c3, z[2], &Wp, &tau_t, &cnt);
                    if (rc.launch_forced >= 0) transport(&rc, (uint32_t)pkt, pp, nn3, c3, Wp, tau_t, 0, batch, &cnt);
                    else if (rc.evcount) rc.evcount[pkt] = 0;
                    out->counters.events += cnt.events;
                    out->counters.segments_transport += cnt.segments_transport;
                    out->counters.segments_peel += cnt.segments_peel;
                    out->counters.packets_escaped += cnt.packets_escaped;
                    out->counters.packets_absorbed += cnt.packets_absorbed;
                    out->counters.packets_surface += cnt.packets_surface;
                    out->counters.packets_stuck += cnt.packets_stuck;
                    out->counters.escaped_weight += cnt.escaped_weight;
                }
            }
        }
    }
    chan_free(&ch);
    geom_free(&G);
    return 0;
}

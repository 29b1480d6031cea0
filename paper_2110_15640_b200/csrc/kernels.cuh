// kernels.cuh -- the packet kernels of libgcmcrt (sm_100a): opacity staging (A0/A1), emission CDF (A2),
// persistent-thread transport with warp-level refill (A3-A6, A8), the separate peel-off ray integrator with
// shared-memory flux bins (A7, A9) and the normalisation (A10).  See DESIGN.md for the data layout.
#pragma once
#include "ray.cuh"
#include "sort.cuh"

namespace gcmcrt {

constexpr int kMaxObs = 32;
constexpr int kMaxBatches = 64;
constexpr int kTransportThreads = 256;
constexpr int kPeelThreads = 256;

// Packed cell id: i | j << 10 | k << 20  (nlev, nlat <= 1024, nlon <= 2048)
__device__ __forceinline__ uint32_t pack_cell(int i, int j, int k) { return uint32_t(i) | uint32_t(j) << 10 | uint32_t(k) << 20; }
__device__ __forceinline__ void unpack_cell(uint32_t c, int& i, int& j, int& k) { i = c & 1023; j = (c >> 10) & 1023; k = c >> 20; }

enum EventKind : uint32_t { EV_MEDIUM = 0, EV_EMIT = 1, EV_SURFACE = 2 };

struct EventBuf;
__device__ __forceinline__ void write_event(const EventBuf& ev, unsigned int slot, float px, float py, float pz, float W,
                                            float nx, float ny, float nz, uint32_t m_inter, uint32_t cellp, uint32_t meta,
                                            uint32_t pkt, float4 prop);

// Event records written by the transport kernels, consumed by the peel kernel and by the next generation: one
// 64-byte, 64-byte-aligned record per event = two whole 32 B sectors, so that reading records through the sort
// permutation moves no byte it does not use.
struct EventBuf {
    float4* rec;  // [cap][4]:
                  //   [0] px py pz W             packet weight before the event
                  //   [1] nx ny nz 0             n = incoming direction (medium) or surface normal
                  //   [2] m_inter cell meta pkt  (bit patterns) interactions completed before this event; packed cell;
                  //                              meta = kind | batch << 2 | chan_run << 8; packet id
                  //   [3] omega P_gas g kappa    the cell's scattering properties (medium events; zeros otherwise)
                  // The record is the peel kernel's input AND the packet's full state at the event: the wavefront
                  // kernels continue packets from it.
    unsigned int* count;
    unsigned int cap;
    unsigned int soft_cap;
    // first half of the counting sort by (channel, cell) (sort.cuh), done while the record is written: the key is kept
    // and its histogram bin counted, so that the sort itself is one scan and one scatter.  NULL when no peel follows.
    unsigned int* keys;   // [cap]
    unsigned int* hist;   // [c_fold * ncell], zeroed by the host before the pass; NULL: the host runs ev_hist_kernel
                          // instead (emission: events pile up in a few bright cells and the contended atomics are
                          // cheaper in a kernel of their own than inside the emit / interact kernels)
    const int* chan_lo;   // device: first channel of the pass (PassCtrl::chan_lo)
    int c_fold, nlev, nlat, ncell;
    int lev_shift, nlg, bins_per_chan;   // the key's second part is column * nlg + (i >> lev_shift): cells (shift 0),
                                         // groups of levels, or whole columns (nlg = 1)
};

__device__ __forceinline__ void write_event(const EventBuf& ev, unsigned int slot, float px, float py, float pz, float W,
                                            float nx, float ny, float nz, uint32_t m_inter, uint32_t cellp, uint32_t meta,
                                            uint32_t pkt, float4 prop)
{
    GCMCRT_CHECK(slot < ev.cap);
    float4* r = ev.rec + 4 * (size_t)slot;
    r[0] = make_float4(px, py, pz, W);
    r[1] = make_float4(nx, ny, nz, 0.f);
    r[2] = make_float4(__uint_as_float(m_inter), __uint_as_float(cellp), __uint_as_float(meta), __uint_as_float(pkt));
    r[3] = prop;
    if (ev.keys) {
        const int i = cellp & 1023, j = (cellp >> 10) & 1023, k = cellp >> 20;
        const unsigned int chan = (unsigned int)min(max(int(meta >> 8) - *ev.chan_lo, 0), ev.c_fold - 1);
        const unsigned int col = (unsigned int)(k * ev.nlat + j);
        const unsigned int key = chan * (unsigned int)ev.bins_per_chan + col * (unsigned int)ev.nlg + (ev.nlg > 1 ? (unsigned int)(i >> ev.lev_shift) : 0u);
        GCMCRT_CHECK(i < ev.nlev && j < ev.nlat && key < (unsigned int)ev.c_fold * (unsigned int)ev.bins_per_chan);
        ev.keys[slot] = key;
        if (ev.hist) atomicAdd(ev.hist + key, 1u);
    }
}

// Packets suspended because the event buffer filled up; resumed by the next pass.
struct SuspBuf {
    float4* s0;  // px py pz W
    float4* s1;  // nx ny nz cell
    uint4* s2;   // chan_run pkt m_inter nev|kind<<28
    unsigned int* count;
    unsigned int* taken;
    unsigned int cap;   // entries allocated: a park beyond it is dropped and counted as a stuck packet (the host sizes the
                        // list so that this cannot happen and reports an error if the count ever exceeds it)
};

struct PassCtrl;
struct SuspPair {   // the two suspended lists; which one a pass reads is part of the pass plan (PassCtrl::cur)
    SuspBuf b[2];
};
// field-by-field selects: indexing the kernel parameter with a run-time value would copy it to the stack
__device__ __forceinline__ SuspBuf susp_select(const SuspPair& p, int which)
{
    SuspBuf s;
    s.s0 = which ? p.b[1].s0 : p.b[0].s0; s.s1 = which ? p.b[1].s1 : p.b[0].s1; s.s2 = which ? p.b[1].s2 : p.b[0].s2;
    s.count = which ? p.b[1].count : p.b[0].count; s.taken = which ? p.b[1].taken : p.b[0].taken;
    s.cap = which ? p.b[1].cap : p.b[0].cap;
    return s;
}

struct DevCounters {
    unsigned long long events, seg_transport, seg_peel, escaped, absorbed, surface, stuck, rays_peel;
    double escaped_weight;
};

// Pass control, device-resident.  A run is a sequence of passes (fresh packets whose events fit the event buffer, then
// the peel-off of those events); everything that changes from pass to pass lives here and is read by the kernels, so
// that the host never has to look at it: pass_begin_kernel / pass_end_kernel (below) are the loop's bookkeeping and
// the loop itself is a conditional WHILE node of a CUDA graph (gcmcrt.cu).
constexpr int kMaxGen = 30;
struct alignas(128) PassCtrl {
    // -- counters the packet kernels update with atomics (zeroed by pass_begin_kernel)
    unsigned int ev_count;
    unsigned int susp_count[2];
    unsigned int susp_taken[2];
    unsigned int pad0;
    unsigned long long work_counter;   // next fresh item (persistent-only transport); kept from pass to pass
    unsigned long long ray_counter;
    unsigned int gen_mark[kMaxGen + 2];   // event-buffer offsets of the wavefront generations of this pass
    // -- the plan of the current pass (written by pass_begin_kernel, read-only for the packet kernels)
    alignas(128) unsigned long long item0;   // first fresh packet item of this pass (item = chan_run * n_pkt + packet offset)
    unsigned int n_fresh;              // fresh packets of this pass (wavefront transport)
    int cur;                           // suspended list this pass resumes from; it parks into the other one
    int chan_lo;                       // first channel this pass draws fresh packets from (sort key window)
    int done, error;                   // error: 1 suspended-list overflow, 2 pass limit
    // -- loop state (control kernels only)
    unsigned long long batch, ev_seen, pk_seen, leftover, passes;
};

struct PassPlan {   // constants of one run's pass loop
    unsigned long long total_items, susp_cap, max_passes, batch0;
    unsigned int n_pkt, ev_cap;
    int n_gen;          // wavefront generations per pass (0: the persistent kernel draws the fresh packets itself)
    int n_chan_run;
};

// start of a run (one per Doppler observer run): loop state to its initial values; the pass count carries on
__global__ void run_begin_kernel(PassCtrl* c, const PassPlan p)
{
    const unsigned long long passes = c->passes;
    const int error = c->error;
    *c = PassCtrl{};
    c->passes = passes; c->error = error;
    c->batch = p.batch0;
}

// end of a generation: the events written so far (a kernel, not a 4-byte copy: a memcpy node inside the loop body of
// the graph costs tens of microseconds)
__global__ void gen_mark_kernel(PassCtrl* c, int m) { c->gen_mark[m] = c->ev_count; }

__global__ void pass_begin_kernel(PassCtrl* c, const PassPlan p)
{
    const int nxt = 1 - c->cur;
    c->ev_count = 0; c->ray_counter = 0;
    c->susp_count[nxt] = 0; c->susp_taken[0] = 0; c->susp_taken[1] = 0;
    for (int m = 0; m < kMaxGen + 2; ++m) c->gen_mark[m] = 0;
    unsigned long long nf = 0;
    if (p.n_gen > 0 && !c->done) {
        // fresh packets sized so that all their events fit the event buffer (the ratio events / packet is learnt from
        // the passes already run); a pass that inherited a long suspended list only drains it
        const unsigned long long room = p.total_items - c->item0;
        nf = c->leftover > p.ev_cap / 2 ? 0ull : min(min(c->batch, (unsigned long long)(p.ev_cap / 2)), room);
    }
    c->n_fresh = (unsigned int)nf;
    c->chan_lo = (int)min(c->item0 / max(p.n_pkt, 1u), (unsigned long long)p.n_chan_run);
}

// end of a pass: what the host loop used to do after reading the counters back.  use_handle: the loop is a conditional
// WHILE node and this kernel sets its condition; else the host reads `done`.
__global__ void pass_end_kernel(PassCtrl* c, const PassPlan p, cudaGraphConditionalHandle handle, int use_handle)
{
    const int cur = c->cur, nxt = 1 - cur;
    if (p.n_gen > 0) {
        c->item0 += c->n_fresh;
        c->ev_seen += min(c->ev_count, p.ev_cap);
        c->pk_seen += c->n_fresh;
        if (c->pk_seen > 0) {   // next batch: 85 % of the buffer at the ratio seen so far
            const double ratio = fmax(0.25, double(c->ev_seen) / double(c->pk_seen));
            c->batch = max(1024ull, (unsigned long long)(0.85 * double(p.ev_cap) / ratio));
        }
    } else {
        c->item0 = min(c->work_counter, p.total_items);
    }
    c->leftover = c->susp_count[nxt];
    if (c->leftover > p.susp_cap) c->error = 1;
    c->passes += 1;
    c->done = (c->item0 >= p.total_items && c->leftover == 0) ? 1 : 0;
    if (!c->done && c->passes >= p.max_passes) c->error = 2;
    if (!c->done && !c->error) { c->susp_count[cur] = 0; c->cur = nxt; }
    if (use_handle) cudaGraphSetConditional(handle, (c->done || c->error) ? 0u : 1u);
}

struct RunConst {
    GeomParams geom;
    const float* alpha;    // [n_chan_tab][ncol][col_stride] extinction (m^-1), guard-padded columns (ray.cuh)
    const float4* prop;    // [n_chan_tab][ncell] omega, P_gas, g, k_abs_eff
    const double* Lcum;    // emission: [n_chan_tab][ncell] running luminosity inside the cell's column
    const double* Lcol;    // emission: [n_chan_tab][ncol] luminosity of the columns before (emis_cum())
    const double* Lcell;   // emission, xi > 0 only
    const double* Ltot;    // emission: [n_chan_tab]
    const int* guide;      // emission: [n_chan_tab][kEmisGuide] search brackets of the CDF (emis_guide_kernel)
    uint32_t chan_key0;    // global channel index of table row 0 (Philox key)
    int chan_begin;        // first table row of this run
    int n_chan_run;
    uint32_t pkt_begin, n_pkt;
    unsigned long long N;  // packets_per_channel
    unsigned long long seed;
    int mode;              // 0 albedo, 1 emission
    int max_events, scatter_on;
    int survival_bias;             // Sect. 4.4: forced scattering with W <- W omega
    float roulette_w_min, roulette_survive;   // Sect. 4.5: Russian roulette below the weight threshold (0 = off)
    int cloud_phase;               // 0 HG (Eq. 7-8), 1 two-term HG (Eq. 10, g1 = g, g2 = -g/2, alpha = 1 - g2^2), 2 Draine (Eq. 9)
    const float* alpha2;           // continuous absorption: [n_chan][ncol][col_stride] pairs (alpha_sca, alpha_abs), or NULL
    int forced_scatter;            // Sect. 4.2: 1 = forced first scattering of albedo packets, 2 = every flight forced
    float stretch, inv_stretch;    // Sect. 4.2, path length stretching: flights from a e^{-a tau}, a = stretch (1 = off), 1 / a
    // Sect. 5.1 with multiple scattering (L259, N12): packets start on transit chords toward observer `obs_first`
    // instead of on the star-facing disc; every peel-off of packet i enters the flux with the factor
    // -W_ld,i b_i dOmega (chord_scale(): a function of the packet's launch block, recomputed where it is needed)
    int launch_chord;
    float launch_dir[3];           // direction of the first flight: -star (albedo) or the observer (chords)
    float tr_ex[3], tr_ey[3];      // sky-plane frame of the chords' observer (C19)
    float tr_star_radius, tr_planet_x, tr_planet_y, tr_ld_c1, tr_ld_c2, tr_domega;
    float surface_albedo;
    double xi;
    int n_batches;
    int n_obs_run, obs_first, n_obs_total;
    float star[3], e1[3], e2[3];
    float obs[kMaxObs][3];
    float img_ex[kMaxObs][3], img_ey[kMaxObs][3];
    float tau_cut;
    int npix;
    // outputs
    double* flux;          // [n_chan_run][n_obs_total][n_batches]
    float* image;          // nullable
    float* contrib;        // nullable [n_chan_run][n_obs_total][2][ncell]: Eq. 32 numerators (thermal, scattered)
    uint32_t* event_count; // nullable [n_chan_run][n_pkt]
    DevCounters* counters;
    unsigned long long* work_counter;   // next fresh packet item
    unsigned long long* ray_counter;    // next peel ray of this pass
    const PassCtrl* ctrl;               // the pass plan (device)
    // exact-division constants floor(2^64 / d) for d = N, n_pkt, n_obs_run (device_common.cuh div_magic)
    unsigned long long magic_N, magic_npkt, magic_nobs;
    // warp scheduling thresholds (lanes waiting before the warp leaves the radial march to serve them)
    int t_service;   // transport: finished / idle / event lanes
    int t_lateral;   // both kernels: lanes parked at a cone or half-plane
    int p_refill;    // peel: finished / idle lanes
};

// ---------------------------------------------------------------------------------------------------------
// A0 / A1: opacity staging.  One thread per (channel, cell); coalesced along the radial index.
// ---------------------------------------------------------------------------------------------------------
struct StageParams {
    int n_chan, ncell, nlev, nlat, nlon;
    int c_begin, c_end;    // channels to stage (a part of a run stages its own channels only); the tables hold n_chan
    const float *k_abs, *k_ray, *k_cld, *g_cld, *rho;
    float* alpha;          // [n_chan][ncol][col_stride], zero-filled by the host before the launch (guard entries)
    float* alpha2;         // continuous absorption: the same layout with (alpha_sca, alpha_abs) pairs, or NULL
    long long alpha_stride;
    int col_stride;
    float4* prop;
    // k_abs from (T, log10 p) node tables instead of a per-cell table (the on-GPU opacity interpolator, Sect. 7):
    // k_abs(c, cell) = bilinear interpolation of node[c][nT][nP] at the cell's (T, log10 p), clamped to the table
    const float* node;     // [n_chan][nT][nP] or NULL
    const int2* node_idx;  // [ncell] (iT, iP) of the lower-left node
    const float2* node_w;  // [ncell] weights of the upper nodes
    int nT, nP;
    // Doppler (A1): per-cell line-of-sight velocity of this observer, per-channel 1/ln(lambda ratio)
    int doppler, halfwidth;
    const float* vlos;   // [ncell] for the current observer
    const float* reff;   // [n_chan]
};

__global__ void __launch_bounds__(256) vlos_kernel(int nlev, int nlat, int nlon, const float* __restrict__ u,
                                                   const float* __restrict__ v, const float* __restrict__ w, float Omega,
                                                   const float* __restrict__ rc, const float* __restrict__ thc,
                                                   const float* __restrict__ phc, float ox, float oy, float oz,
                                                   float* __restrict__ vlos)
{
    // Eq. 33 in vector form (C13): v_LOS = -(u phi^ - v theta^ + w r^ + Omega r sin(theta) phi^) . o^ at the cell centre
    const int cell = blockIdx.x * blockDim.x + threadIdx.x;
    const int ncell = nlev * nlat * nlon;
    if (cell >= ncell) return;
    const int i = cell % nlev, j = (cell / nlev) % nlat, k = cell / (nlev * nlat);
    float st, ct, sp, cp;
    sincosf(thc[j], &st, &ct);
    sincosf(phc[k], &sp, &cp);
    const float ue = (u ? u[cell] : 0.0f) + Omega * rc[i] * st;
    const float vn = v ? v[cell] : 0.0f, wu = w ? w[cell] : 0.0f;
    const float Vx = ue * (-sp) - vn * (ct * cp) + wu * (st * cp);
    const float Vy = ue * cp - vn * (ct * sp) + wu * (st * sp);
    const float Vz = vn * st + wu * ct;
    vlos[cell] = -(Vx * ox + Vy * oy + Vz * oz);
}

// per cell: position of (T, log10 p) in the uniform node grid
__global__ void __launch_bounds__(256) node_coeff_kernel(int ncell, const float* __restrict__ T, const float* __restrict__ p_cell,
                                                         float T0, float dT, float lp0, float dlp, int nT, int nP,
                                                         int2* __restrict__ idx, float2* __restrict__ w)
{
    const int cell = blockIdx.x * blockDim.x + threadIdx.x;
    if (cell >= ncell) return;
    const float ft = fminf(fmaxf((T[cell] - T0) / dT, 0.0f), float(nT - 1) - 1e-4f);
    const float fp = fminf(fmaxf((log10f(p_cell[cell]) - lp0) / dlp, 0.0f), float(nP - 1) - 1e-4f);
    const int it = int(ft), ip = int(fp);
    idx[cell] = make_int2(it, ip);
    w[cell] = make_float2(ft - float(it), fp - float(ip));
}

__device__ __forceinline__ float stage_kabs(const StageParams& p, int c, int cell)
{
    if (p.node) {
        const int2 id = __ldg(p.node_idx + cell);
        const float2 w = __ldg(p.node_w + cell);
        const float* nd = p.node + ((size_t)c * p.nT + id.x) * p.nP + id.y;
        const float a00 = __ldg(nd), a01 = __ldg(nd + 1), a10 = __ldg(nd + p.nP), a11 = __ldg(nd + p.nP + 1);
        return (1.0f - w.x) * ((1.0f - w.y) * a00 + w.y * a01) + w.x * ((1.0f - w.y) * a10 + w.y * a11);
    }
    return __ldg(p.k_abs + (long long)c * p.ncell + cell);
}

// grid = (cell tiles, channels): a thread stages one cell of one channel; consecutive lanes read consecutive cells of
// the caller's tables and write consecutive prop records (alpha: consecutive inside a column).  HBM-bound: per
// (channel, cell) 4-16 B of tables in, 4 B alpha + 16 B prop out.
__global__ void __launch_bounds__(256) stage_kernel(const StageParams p)
{
    const int cell = blockIdx.x * blockDim.x + threadIdx.x;
    if (cell >= p.ncell) return;
    const int col = cell / p.nlev;   // once per thread: the thread then loops over channels
    const int i = cell - col * p.nlev;
    const float rho = __ldg(p.rho + cell);
    float dn_cell = 0.0f;
    if (p.doppler && p.n_chan > 1) dn_cell = -__ldg(p.vlos + cell) * (1.0f / 299792458.0f);
    // four channels per round, all their loads issued before the first store: the kernel lives on bytes in flight
    constexpr int U = 4;
    for (int c0 = p.c_begin + blockIdx.y * U; c0 < p.c_end; c0 += gridDim.y * U) {
        float ka[U], kr[U], kc[U], gg[U];
#pragma unroll
        for (int q = 0; q < U; ++q) {
            const int c = min(c0 + q, p.c_end - 1);
            const long long t = (long long)c * p.ncell + cell;
            if (p.doppler && p.n_chan > 1) {
                // Eq. 34: lambda_eff = lambda_0 (1 - v/c) -> index offset dn = -v/c / ln(lambda_{n+1}/lambda_n), C14
                float dn = dn_cell * p.reff[c];
                dn = fminf(fmaxf(dn, -float(p.halfwidth)), float(p.halfwidth));
                // integer and fractional part of dn apart: c + dn in fp32 would lose the fraction at c ~ 1e5 and make
                // the result depend on where a wavelength batch starts
                const float fl = floorf(dn);
                int lo = c + int(fl);
                float f = dn - fl;
                if (lo < 0) { lo = 0; f = 0.0f; }
                if (lo > p.n_chan - 2) { lo = p.n_chan - 2; f = 1.0f; }
                const float k0 = stage_kabs(p, lo, cell), k1 = stage_kabs(p, lo + 1, cell);
                ka[q] = (1.0f - f) * k0 + f * k1;
            } else {
                ka[q] = stage_kabs(p, c, cell);
            }
            kr[q] = p.k_ray ? __ldg(p.k_ray + t) : 0.0f;
            kc[q] = p.k_cld ? __ldg(p.k_cld + t) : 0.0f;
            gg[q] = p.g_cld ? __ldg(p.g_cld + t) : 0.0f;
        }
#pragma unroll
        for (int q = 0; q < U; ++q) {
            const int c = c0 + q;
            if (c >= p.c_end) break;
            const long long t = (long long)c * p.ncell + cell;
            const float ks = kr[q] + kc[q];
            const float kext = ka[q] + ks;
            // guard-padded column layout of the marcher: [chan][col][col_stride], level i at offset 1 + i
            const size_t at = (size_t)c * p.alpha_stride + (size_t)col * p.col_stride + 1 + i;
            p.alpha[at] = rho * kext;
            float omega = kext > 0.0f ? ks / kext : 0.0f;
            if (p.alpha2) {   // continuous absorption (Eq. 12): flights march (alpha_sca, alpha_abs); every interaction drawn
                              // from alpha_sca is a scattering, which the event code reads as omega = 1
                reinterpret_cast<float2*>(p.alpha2)[at] = make_float2(rho * ks, rho * ka[q]);
                omega = ks > 0.0f ? 1.0f : 0.0f;
            }
            p.prop[t] = make_float4(omega, ks > 0.0f ? kr[q] / ks : 0.0f, gg[q], ka[q]);
        }
    }
}

// ---------------------------------------------------------------------------------------------------------
// A2: emission luminosities (Eq. 27), tau_vert cut (L210, C15) and the running sum used as CDF (Eq. 13).
// ---------------------------------------------------------------------------------------------------------
struct EmisParams {
    int n_chan, nlev, nlat, nlon, ncell;
    const float* alpha;
    long long alpha_stride;
    int col_stride;
    const float4* prop;
    const float *rho, *T;
    const double* lambda;   // [n_chan]
    const double *r_edges, *cth_edges, *ph_edges;  // fp64 geometry for the volumes
    double tau_vert_max;
    double* Lcell;  // [n_chan][ncell] L_i, or NULL (kept for the weights of the composite bias, xi > 0)
    double* Lcum;   // [n_chan][ncell] column-local running sum
    double* Lcol;   // [n_chan][nlat * nlon] column totals (emis_col_kernel), then the sums of the columns before (emis_colscan_kernel)
    double* Ltot;
};

__device__ __forceinline__ double planck_lambda(double lam, double T)
{
    const double h = 6.62607015e-34, c = 299792458.0, kb = 1.380649e-23;
    const double x = h * c / (lam * kb * T);
    return 2.0 * h * c * c / (lam * lam * lam * lam * lam) / expm1(x);
}

// 1 / x for a positive, finite, normal x to ~1 ulp: the 20-bit hardware seed and two Newton steps (7 instructions; the
// IEEE division is ~30 with its special-case path).  The emission kernel divides twice per (channel, cell).
__device__ __forceinline__ double rcp_pos_f64(double x)
{
    double r;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
    r = fma(r, fma(-x, r, 1.0), r);
    r = fma(r, fma(-x, r, 1.0), r);
    return r;
}

__device__ __forceinline__ double warp_incl_scan_f64(double v)
{
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const double n = __shfl_up_sync(kFullMask, v, o);
        if (lane_id() >= o) v += n;
    }
    return v;
}

// The CDF is stored in two levels, so that no thread waits for another column:
//   Lcum[c][cell]  running sum of L_i inside the cell's own column (from its lowest level up to the cell, inclusive),
//   Lcol[c][col]   sum of the columns before `col` (exclusive), Ltot[c] the channel's total,
// and the running sum of Eq. 13 at a cell is emis_cum() = Lcol[c][col] + Lcum[c][cell].  It never decreases from one
// cell to the next: inside a column the same offset is added to a non-decreasing sequence, and Lcol[col + 1] is
// fl(Lcol[col] + total(col)) by construction (emis_colscan_kernel adds the totals in column order), total(col) being
// the column's last local value.
__device__ __forceinline__ double emis_cum(const double* __restrict__ cum_c, const double* __restrict__ col_c, int nlev, int cell)
{
    return col_c[cell / nlev] + cum_c[cell];
}

// First cell whose running luminosity exceeds x, searched in [lo, hi] (Eq. 13), in two levels: the column first -- the
// running sum at a column's last cell IS the next column's offset (the channel's total after the last column) -- then
// the cell inside it, with the column's offset loaded once.  Both levels evaluate emis_cum() > x, so the result is the
// cell a search over emis_cum() alone finds.
__device__ __forceinline__ int emis_search(const double* __restrict__ cum_c, const double* __restrict__ col_c, double Ltot,
                                           int nlev, int ncol, int lo, int hi, double x)
{
    int clo = lo / nlev, chi = hi / nlev;
    while (clo < chi) {
        const int cmid = (clo + chi) >> 1;
        const double end = cmid + 1 < ncol ? col_c[cmid + 1] : Ltot;   // == emis_cum(last cell of column cmid)
        if (end > x) chi = cmid; else clo = cmid + 1;
    }
    const double off = col_c[clo];
    lo = max(lo, clo * nlev); hi = min(hi, clo * nlev + nlev - 1);
    while (lo < hi) {
        const int mid = (lo + hi) >> 1;
        if (off + cum_c[mid] > x) hi = mid; else lo = mid + 1;
    }
    return lo;
}

// One warp per (channel, column), lanes along the column (coalesced alpha / prop reads; NCH = chunks of 32 levels),
// blockIdx.y = channel, the warps of a CTA stride through the channel's columns.  A warp loads every input of its
// column up front, finds the depth cut (radial optical depth from the top, C15), computes L_i (Eq. 27), scans it and
// writes the column-local running sum and the column total: no barrier and no dependence between columns, so the SM
// hides one column's latency behind the others'.  HBM traffic per (channel, cell): 4 B alpha + 16 B prop in, 8 B out
// (T, rho stay in L2 across channels).
constexpr int kEmisThreads = 256;
template <int NCH>
__global__ void __launch_bounds__(kEmisThreads) emis_col_kernel(const EmisParams p)
{
    extern __shared__ double emis_sm[];
    double* dr = emis_sm;                 // [nlev] R_{i+1} - R_i
    double* dr3 = dr + p.nlev;            // [nlev] (R_{i+1}^3 - R_i^3) / 3
    const int lane = lane_id(), wid = threadIdx.x >> 5;
    for (int i = threadIdx.x; i < p.nlev; i += blockDim.x) {
        const double r0 = p.r_edges[i], r1 = p.r_edges[i + 1];
        dr[i] = r1 - r0;
        dr3[i] = (r1 * r1 * r1 - r0 * r0 * r0) / 3.0;
    }
    __syncthreads();
    const int ncol = p.nlat * p.nlon;
    for (int c = blockIdx.y; c < p.n_chan; c += gridDim.y) {
        const double lam = p.lambda[c];
        const double hck = 6.62607015e-34 * 299792458.0 / (lam * 1.380649e-23);                     // h c / (lambda k)
        const double pre = 4.0 * 3.14159265358979323846 * 2.0 * 6.62607015e-34 * 299792458.0 * 299792458.0 /
                           (lam * lam * lam * lam * lam);                                            // 4 pi 2 h c^2 / lambda^5
        const float* alpha_c = p.alpha + (size_t)c * p.alpha_stride;
        const float4* prop_c = p.prop + (size_t)c * p.ncell;
        double* out = p.Lcum + (size_t)c * p.ncell;
        for (int col = blockIdx.x * (kEmisThreads / 32) + wid; col < ncol; col += gridDim.x * (kEmisThreads / 32)) {
            const size_t cell0 = (size_t)col * p.nlev;
            const float* acol = alpha_c + (size_t)col * p.col_stride + 1;
            float a[NCH], T[NCH];
            double rk[NCH];   // rho kappa_abs: the fp64 product of two fp32 values is exact, as in the oracle's fp64
    #pragma unroll
            for (int m = 0; m < NCH; ++m) {                  // level i = 32 m + lane
                const int i = (m << 5) + lane;
                const bool in = i < p.nlev;
                a[m] = in ? __ldg(acol + i) : 0.0f;
                T[m] = in ? __ldg(p.T + cell0 + i) : 1.0f;
                rk[m] = in ? double(__ldg(p.rho + cell0 + i)) * double(__ldg(&prop_c[cell0 + i].w)) : 0.0;
            }
            // depth cut: cell i is dropped when the radial optical depth of the levels above it exceeds tau_vert_max;
            // suffix sums from the top = column total - inclusive prefix from below
            int i_cut = 0;   // lowest level kept
            if (p.tau_vert_max > 0.0) {
                double incl[NCH], tot = 0.0;
    #pragma unroll
                for (int m = 0; m < NCH; ++m) {
                    const int i = (m << 5) + lane;
                    const double d = i < p.nlev ? double(a[m]) * dr[i] : 0.0;
                    incl[m] = tot + warp_incl_scan_f64(d);
                    tot = __shfl_sync(kFullMask, incl[m], 31);
                }
    #pragma unroll
                for (int m = 0; m < NCH; ++m) {
                    const int i = (m << 5) + lane;
                    const unsigned mc = __ballot_sync(kFullMask, i < p.nlev && (tot - incl[m]) > p.tau_vert_max);
                    if (mc) i_cut = (m << 5) + 32 - __clz(mc);   // highest cut level + 1 (the sum only grows downward)
                }
            }
            const int j = col % p.nlat, k = col / p.nlat;
            const double ang = (p.cth_edges[j] - p.cth_edges[j + 1]) * (p.ph_edges[k + 1] - p.ph_edges[k]);
            double run = 0.0;
    #pragma unroll
            for (int m = 0; m < NCH; ++m) {
                const int i = (m << 5) + lane;
                double Li = 0.0, sum = run;
                if ((m << 5) + 32 > i_cut && (m << 5) < p.nlev) {   // warp-uniform: a chunk wholly below the cut holds no luminosity
                    if (i < p.nlev && i >= i_cut) {
                    const double e = expm1(hck * rcp_pos_f64(double(T[m])));     // +inf in the far Wien tail: L_i = 0
                    Li = e < 1e300 ? pre * dr3[i] * ang * rk[m] * rcp_pos_f64(e) : 0.0;
                }
                    sum = run + warp_incl_scan_f64(Li);
                    run = __shfl_sync(kFullMask, sum, 31);
                }
                if (i < p.nlev) {
                    if (p.Lcell) p.Lcell[(size_t)c * p.ncell + cell0 + i] = Li;
                    out[cell0 + i] = sum;
                }
            }
            if (lane == 0) p.Lcol[(size_t)c * ncol + col] = run;
        }
    }
}

// Column offsets of the two-level CDF: one warp per channel turns the column totals emis_col_kernel left in Lcol into
// the sums of the columns before each (in place) and writes the channel's total.  The totals are added one by one in
// column order -- every lane runs the same chain over the 32 totals of a chunk -- so that
// Lcol[col + 1] == fl(Lcol[col] + total(col)) exactly, which is what keeps emis_cum() monotonic across columns.
__global__ void __launch_bounds__(128) emis_colscan_kernel(int n_chan, int ncol, double* __restrict__ Lcol, double* __restrict__ Ltot)
{
    const int c = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = lane_id();
    if (c >= n_chan) return;
    double* col = Lcol + (size_t)c * ncol;
    double carry = 0.0;
    for (int col0 = 0; col0 < ncol; col0 += 32) {
        const double v = col0 + lane < ncol ? col[col0 + lane] : 0.0;
        double excl = 0.0;
#pragma unroll
        for (int w = 0; w < 32; ++w) {
            if (w == lane) excl = carry;
            carry += __shfl_sync(kFullMask, v, w);
        }
        if (col0 + lane < ncol) col[col0 + lane] = excl;
    }
    if (lane == 0) Ltot[c] = carry;
}

// Guide table of the emission CDF: guide[c][g] = first cell whose running luminosity exceeds (g / kEmisGuide) L_tot.
// A packet's search (Eq. 13) then starts from the bracket [guide[g], guide[g+1]] of its own g = floor(frac * kEmisGuide)
// -- a few cells in the bright part of the atmosphere instead of 17 dependent loads over the whole table -- and finds
// the same cell as the full search (the bracket contains it by monotonicity of frac -> frac * L_tot in fp64).
constexpr int kEmisGuide = 4096;

__global__ void __launch_bounds__(256) emis_guide_kernel(int n_chan, int ncell, int nlev, const double* __restrict__ Lcum,
                                                         const double* __restrict__ Lcol, const double* __restrict__ Ltot,
                                                         int* __restrict__ guide)
{
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= (long long)n_chan * kEmisGuide) return;
    const int c = int(t / kEmisGuide), gi = int(t % kEmisGuide);
    const double x = double(gi) / double(kEmisGuide) * Ltot[c];
    guide[t] = emis_search(Lcum + (size_t)c * ncell, Lcol + (size_t)c * (ncell / nlev), Ltot[c], nlev, ncell / nlev, 0, ncell - 1, x);
}

// ---------------------------------------------------------------------------------------------------------
// Transit chords (Sect. 5.1, Eq. 20-23): launch block (zeta0, zeta1) -> impact parameter b uniform in [R_p0, R_TOA]
// (Eq. 21 carries the factor b_i), azimuth around the limb, limb-darkening weight of the stellar disc point behind it.
// ---------------------------------------------------------------------------------------------------------
__device__ __forceinline__ void chord_point(const RunConst& rc, float z0, float z1, float& b, float& X, float& Y, float& W)
{
    b = fmaf(z0, rc.geom.Rtoa - rc.geom.R0, rc.geom.R0);
    float sp, cp;
    sincospif(2.0f * z1, &sp, &cp);
    X = b * cp; Y = b * sp;
    W = 1.0f;
    if (rc.tr_star_radius > 0.f) {                         // Eq. 22-23
        const float sx = (rc.tr_planet_x + X) / rc.tr_star_radius, sy = (rc.tr_planet_y + Y) / rc.tr_star_radius;
        const float rho2 = fmaf(sx, sx, sy * sy);
        const float mu1 = 1.0f - sqrtf(fmaxf(0.f, 1.0f - rho2));
        W = rho2 >= 1.0f ? 0.f : 1.0f - rc.tr_ld_c1 * mu1 - rc.tr_ld_c2 * mu1 * mu1;
    }
}
// the chord's start on the star side of the TOA sphere
__device__ __forceinline__ void chord_start(const RunConst& rc, float b, float X, float Y, float& px, float& py, float& pz)
{
    const float Rt = rc.geom.Rtoa, h = sqrtf(fmaxf(0.f, (Rt - b) * (Rt + b)));
    px = X * rc.tr_ex[0] + Y * rc.tr_ey[0] - h * rc.launch_dir[0];
    py = X * rc.tr_ex[1] + Y * rc.tr_ey[1] - h * rc.launch_dir[1];
    pz = X * rc.tr_ex[2] + Y * rc.tr_ey[2] - h * rc.launch_dir[2];
}
// what a peel-off of packet (ckey, pkt) adds to the chord's term of Eq. 21: -W_ld b dOmega (reading N12)
__device__ __forceinline__ float chord_scale(const RunConst& rc, uint32_t ckey, uint32_t pkt)
{
    const Zeta4 z = zeta_block(rc.seed, ckey, pkt, 0, 0);
    float b, X, Y, W;
    chord_point(rc, z.z0, z.z1, b, X, Y, W);
    return -W * b * rc.tr_domega;
}

// ---------------------------------------------------------------------------------------------------------
// Scattering physics (A8), fp32.
// ---------------------------------------------------------------------------------------------------------
// Eq. 6 as repaired (C7): q = 4 zeta - 2, u = cbrt(q + sqrt(1 + q^2)), cos = u - 1/u
__device__ __forceinline__ float sample_rayleigh(float z)
{
    const float q = fmaf(4.0f, z, -2.0f);
    const float u = cbrtf(q + sqrtf(fmaf(q, q, 1.0f)));
    return u - 1.0f / u;
}
// Eq. 8; |g| < 1e-3 -> Eq. 2 (C8)
__device__ __forceinline__ float sample_hg(float g, float z)
{
    if (fabsf(g) < 1e-3f) return fmaf(2.0f, z, -1.0f);
    const float t = (1.0f - g * g) / (1.0f - g + 2.0f * g * z);
    return (1.0f + g * g - t * t) / (2.0f * g);
}
// Cloud scatterer: HG, or the two-term HG of Eq. 10 whose lobe is picked by zlobe (L152), the part of zeta0 left over
// inside the cloud interval of the partition.
// Draine (2003) phase function, Eq. 9 with the paper's alpha = 0.5 (L146).  Off the hot path (cloud_phase = 2 only):
// plain fp64 bisections in functions of their own, so that the kernels that call them keep their registers.
//   G(g): root of <cos>(G) = G (1 + a (3 + 2 G^2) / 5) / (1 + a (1 + 2 G^2) / 3) = g
//   cosine = zeta-quantile of Eq. 9 through its closed-form CDF (substitution t = 1 + G^2 - 2 G x); the paper's Gibbs
//   sampler is only cited, and one draw per event keeps the stream layout (N10)
__device__ __noinline__ double draine_G(double g)
{
    const double a = 0.5;
    double lo = -1.0, hi = 1.0;
    for (int it = 0; it < 60; ++it) {
        const double G = 0.5 * (lo + hi);
        const double m = G * (1.0 + a * (3.0 + 2.0 * G * G) / 5.0) / (1.0 + a * (1.0 + 2.0 * G * G) / 3.0);
        if (m < g) lo = G; else hi = G;
    }
    return 0.5 * (lo + hi);
}
__device__ __forceinline__ double draine_cdf(double G, double a, double mu)
{
    if (fabs(G) < 1e-3) return (mu + 1.0) + a * (mu * mu * mu + 1.0) / 3.0;
    const double A = 1.0 + G * G, B = 2.0 * G, iB2 = 1.0 / (B * B);
    const double c0 = 1.0 + a * A * A * iB2, c1 = 2.0 * a * A * iB2, c2 = a * iB2 / 3.0;
    const double t = A - B * mu, t0 = A + B, st = sqrt(t), st0 = sqrt(t0);
    return (2.0 / B) * ((c0 / st + c1 * st - c2 * t * st) - (c0 / st0 + c1 * st0 - c2 * t0 * st0));
}
__device__ __noinline__ float sample_draine(float g, float z)
{
    const double a = 0.5, G = draine_G(double(g));
    const double target = double(z) * draine_cdf(G, a, 1.0);
    double lo = -1.0, hi = 1.0;
    for (int it = 0; it < 60; ++it) {
        const double mid = 0.5 * (lo + hi);
        if (draine_cdf(G, a, mid) < target) lo = mid; else hi = mid;
    }
    return float(0.5 * (lo + hi));
}
__device__ __noinline__ float phase_draine(float g, float mu)
{
    const float a = 0.5f, G = float(draine_G(double(g)));
    const float d = 1.0f + G * G - 2.0f * G * mu;
    return (1.0f - G * G) / (1.0f + a * (1.0f + 2.0f * G * G) / 3.0f) * (1.0f + a * mu * mu) / (4.0f * kPi * d * sqrtf(d));
}

__device__ __forceinline__ float sample_cloud(int cloud_phase, float g, float zlobe, float z)
{
    if (cloud_phase == 2) return sample_draine(g, z);
    if (cloud_phase == 1) {
        const float g2 = -0.5f * g, a = 1.0f - g2 * g2;
        return sample_hg(zlobe < a ? g : g2, z);
    }
    return sample_hg(g, z);
}
__device__ __forceinline__ float phase_hg(float g, float mu)
{
    const float d = fmaf(-2.0f * g, mu, 1.0f + g * g);
    const float r = rsqrtf(d);   // d^(-3/2) = r^3: no division, no square root (the peel kernel evaluates this per ray)
    return (1.0f - g * g) * (0.25f / kPi) * (r * r * r);
}
__device__ __forceinline__ float phase_cloud(int cloud_phase, float g, float mu)
{
    if (cloud_phase == 2) return phase_draine(g, mu);
    if (cloud_phase == 1) {
        const float g2 = -0.5f * g, a = 1.0f - g2 * g2;
        return a * phase_hg(g, mu) + (1.0f - a) * phase_hg(g2, mu);
    }
    return phase_hg(g, mu);
}
// C9: rotate n by polar angle acos(ct), azimuth psi = 2 pi zpsi
__device__ __forceinline__ void rotate_dir(float& nx, float& ny, float& nz, float ct, float zpsi)
{
    const float st = sqrtf(fmaxf(0.0f, 1.0f - ct * ct));
    float sp, cp;
    sincospif(2.0f * zpsi, &sp, &cp);
    const float s2 = fmaf(nx, nx, ny * ny);
    float x, y, z;
    if (s2 < 1e-12f) {
        x = st * cp; y = st * sp; z = ct * (nz >= 0.0f ? 1.0f : -1.0f);
    } else {
        const float sq = sqrtf(s2), inv = 1.0f / sq;
        x = st * (nx * nz * cp - ny * sp) * inv + nx * ct;
        y = st * (ny * nz * cp + nx * sp) * inv + ny * ct;
        z = -st * cp * sq + nz * ct;
    }
    const float rn = rsqrtf(fmaf(x, x, fmaf(y, y, z * z)));
    nx = x * rn; ny = y * rn; nz = z * rn;
}

// O6 decision at a medium interaction m (Philox block z of (m, purpose 1)): absorbed, or the polar cosine of the
// scattering angle.  Analog (L192): zeta0 partitions [0, omega P_gas) Rayleigh / [omega P_gas, omega) HG / [omega, 1)
// absorbed (C6).  Survival biasing (Sect. 4.4): always scatters, W <- W omega, zeta0 only picks the scatterer; below
// the roulette threshold (Sect. 4.5) block (m, purpose 2) decides survival with W <- W / p.
__device__ __forceinline__ bool medium_interaction(const RunConst& rc, const float4 pr, const Zeta4& z, uint32_t ckey,
                                                   uint32_t pkt, uint32_t m, float& W, float& ct)
{
    if (rc.survival_bias) {
        if (!(pr.x > 0.0f)) return false;
        W *= pr.x;
        if (rc.roulette_w_min > 0.0f && W < rc.roulette_w_min) {
            const Zeta4 zr = zeta_block(rc.seed, ckey, pkt, m, 2);
            if (zr.z0 >= rc.roulette_survive) return false;
            W /= rc.roulette_survive;
        }
        ct = (z.z0 < pr.y) ? sample_rayleigh(z.z1) : sample_cloud(rc.cloud_phase, pr.z, (z.z0 - pr.y) / (1.0f - pr.y), z.z1);
        return true;
    }
    if (z.z0 >= pr.x) return false;
    const float lo = pr.x * pr.y;
    ct = (z.z0 < lo) ? sample_rayleigh(z.z1) : sample_cloud(rc.cloud_phase, pr.z, (z.z0 - lo) / (pr.x - lo), z.z1);
    return true;
}

// Sect. 4.2 (L179), forced scattering: the "extra raytracing step to calculate the optical depth to the end of the grid
// in the direction of the packet path", lane by lane (the flights it serves are incoherent; the coherent first flights
// of an albedo run have a warp-wide version in wave_first_flight_kernel), then the flight is drawn from the exponential
// law truncated there, the packet keeps the probability 1 - e^-tau_edge of interacting and the uncollided part leaves.
// A ray that ends on a reflecting lower boundary stays analog.
__device__ __noinline__ int ray_tau_to_edge(Ray r, const GeomSmem& s, const float* alpha_c, int maxseg, float& tau)
{
    tau = 0.f;
    int st = RAY_FLYING;
    for (int it = 0; it <= maxseg && st == RAY_FLYING; ++it) {
        st = ray_step(r, s, tau, kInf);
        if (st == RAY_PARK) { ray_lateral(r, s, alpha_c); st = RAY_FLYING; }
    }
    return st;
}
// With path length stretching (rc.stretch = a < 1) this is the hybrid scheme: the stretched law a e^{-a tau} truncated at
// tau_edge.  Returns whether the flight was forced (a flight that was not is stretched by its caller).
__device__ __forceinline__ bool force_flight(const RunConst& rc, const GeomSmem& gs, const Ray& ray, const float* alpha_c,
                                             float& tau_t, float& W, double& escw)
{
    float tau_e;
    const int st = ray_tau_to_edge(ray, gs, alpha_c, rc.geom.maxseg, tau_e);
    if (st == RAY_ESCAPE || (st == RAY_SURFACE && !(rc.surface_albedo > 0.f))) {
        const float pint = -expm1f(-rc.stretch * tau_e);
        if (pint > 0.f) {
            if (st == RAY_ESCAPE) escw += double(W * expf(-tau_e));
            tau_t = -log1pf(-expf(-tau_t) * pint) * rc.inv_stretch;   // the flight's own zeta = e^-tau_t
            W *= pint;
            return true;
        }
    }
    return false;
}

// Path length stretching, the weight of a flight's outcome (p / q of Baes et al. 2016): an interaction after tau carries
// e^{-(1-a) tau} / a, a flight that leaves the medium (top or lower boundary) after tau the ratio e^{-(1-a) tau} of the
// survival probabilities.  a = 1: exactly 1.
__device__ __forceinline__ float stretch_weight(const RunConst& rc, int ray_status, float tau)
{
    if (!(rc.stretch < 1.0f)) return 1.0f;
    const float w = expf(-(1.0f - rc.stretch) * tau);
    return ray_status == RAY_LIMIT ? w * rc.inv_stretch : w;
}

// ---------------------------------------------------------------------------------------------------------
// Transport kernel: persistent threads, one packet per lane, warp-level refill.
// ---------------------------------------------------------------------------------------------------------
// Lane states of the transport kernel.  The warp is a small scheduler: lanes in LS_FLY run the radial march; lanes
// that need anything else wait in their state until enough of them have gathered for the warp to serve that state
// with most lanes active (or until no lane can march any more).
enum LaneState : int {
    LS_IDLE = 0, LS_FLY = 1, LS_EV_MEDIUM = 2, LS_EV_EMIT = 3, LS_EV_SURFACE = 4, LS_DONE = 5,
    LS_PARK = 6,                                         // at a cone / half-plane: ray_lateral() pending
    LS_END_ESC = 7, LS_END_SURF = 8, LS_END_STUCK = 9    // flight over: bookkeeping pending
};

struct Packet {
    Ray ray;
    float tau, tau_t, W;
    float tau_b;   // DUAL: absorption optical depth of the flight in progress (Eq. 12)
    uint32_t chan_run, pkt, m_inter, nev;
    int fl_seg;
};

__device__ __forceinline__ uint32_t batch_of(const RunConst& rc, uint32_t pkt)
{
    return uint32_t(div_magic((unsigned long long)pkt * (unsigned long long)rc.n_batches, rc.N, rc.magic_N));
}

__device__ __forceinline__ void finish_packet(const RunConst& rc, const Packet& pk)
{
    if (rc.event_count) rc.event_count[(size_t)pk.chan_run * rc.n_pkt + (pk.pkt - rc.pkt_begin)] = pk.nev;
}

// DUAL: continuous absorption (Sect. 4.1, Eq. 12): flights march the (alpha_sca, alpha_abs) pair table rc.alpha2, the
// sampled optical depth is spent on alpha_sca and the weight decays by e^-tau_abs at the end of every flight; the staged
// prop records then carry omega = 1, so that the event code below (and the peel kernel) needs no other change.
template <int KSTEPS, bool DUAL>
__global__ void __launch_bounds__(kTransportThreads, 2)
transport_kernel(const __grid_constant__ RunConst rc, const EventBuf ev, const SuspPair susp, const unsigned long long total_items)
{
    extern __shared__ float smem_f[];
    const GeomSmem gs = load_geom(rc.geom, smem_f);
    __syncthreads();
    const int cur_list = rc.ctrl->cur;
    const SuspBuf susp_in = susp_select(susp, cur_list), susp_out = susp_select(susp, 1 - cur_list);

    Packet pk;
    pk.tau = 0.f; pk.tau_t = 0.f; pk.tau_b = 0.f; pk.W = 0.f; pk.chan_run = 0; pk.pkt = 0; pk.m_inter = 0; pk.nev = 0; pk.fl_seg = 0;
    pk.ray = Ray{};
    int st = LS_IDLE;
    auto chan_table = [&](int ctab) {
        return DUAL ? rc.alpha2 + (size_t)ctab * rc.geom.alpha_stride * 2 : rc.alpha + (size_t)ctab * rc.geom.alpha_stride;
    };
    const float* alpha_c = chan_table(0);  // table of this lane's channel
    unsigned long long c_events = 0, c_seg = 0, c_esc = 0, c_abs = 0, c_surf = 0, c_stuck = 0;
    unsigned int c_seg32 = 0;
    double c_escw = 0.0;
    const bool record = rc.n_obs_run > 0;
    bool fresh_left = true;   // warp-uniform: fresh packets may still be available
    const unsigned int n_susp_in = *susp_in.count;
    bool susp_left = n_susp_in > 0;

    for (;;) {
        const unsigned m_fly = __ballot_sync(kFullMask, st == LS_FLY);
        const unsigned m_park = __ballot_sync(kFullMask, st == LS_PARK);
        const unsigned m_ev = __ballot_sync(kFullMask, st >= LS_EV_MEDIUM && st <= LS_EV_SURFACE);
        const unsigned m_end = __ballot_sync(kFullMask, st >= LS_END_ESC);
        unsigned m_idle = __ballot_sync(kFullMask, st == LS_IDLE);
        if (!(fresh_left || susp_left)) {  // nothing to fetch any more: idle lanes are done
            if (st == LS_IDLE) st = LS_DONE;
            m_idle = 0;
        }
        const bool starving = m_fly == 0;
        const int n_service = __popc(m_ev | m_idle | m_end);
        if (n_service >= rc.t_service || (starving && n_service > 0)) {
            c_seg += c_seg32; c_seg32 = 0;
            // ---------------- flights that ended: bookkeeping, then the lane is free ----------------
            if (m_end) {
                if (st >= LS_END_ESC) {
                    if (st == LS_END_ESC) { ++c_esc; c_escw += double(pk.W); }
                    else if (st == LS_END_SURF) ++c_surf;
                    else ++c_stuck;
                    finish_packet(rc, pk);
                    st = (fresh_left || susp_left) ? LS_IDLE : LS_DONE;
                }
                m_idle = __ballot_sync(kFullMask, st == LS_IDLE);
            }
            // ---------------- fetch: resume suspended packets first, then fresh ones ----------------
            if (m_idle) {
                bool need = (st == LS_IDLE);
                if (susp_left) {
                    const unsigned m = __ballot_sync(kFullMask, need);
                    unsigned int base = 0;
                    if (lane_id() == __ffs(m) - 1) base = atomicAdd(susp_in.taken, (unsigned)__popc(m));
                    base = __shfl_sync(kFullMask, base, __ffs(m) - 1);
                    const unsigned int idx = base + rank_in_mask(m);
                    if (need && idx < n_susp_in) {
                        const float4 a = susp_in.s0[idx], b = susp_in.s1[idx];
                        const uint4 c = susp_in.s2[idx];
                        pk.W = a.w; pk.chan_run = c.x; pk.pkt = c.y; pk.m_inter = c.z; pk.nev = c.w & 0x0fffffffu;
                        int i, j, k;
                        unpack_cell(__float_as_uint(b.w), i, j, k);
                        pk.ray.pcx = a.x; pk.ray.pcy = a.y; pk.ray.pcz = a.z; pk.ray.u = 0.f;
                        pk.ray.nx = b.x; pk.ray.ny = b.y; pk.ray.nz = b.z;
                        pk.ray.i = i; pk.ray.j = j; pk.ray.k = k;
                        alpha_c = chan_table(rc.chan_begin + int(pk.chan_run));
                        const uint32_t kind = c.w >> 28;
                        st = kind == EV_MEDIUM ? LS_EV_MEDIUM : (kind == EV_EMIT ? LS_EV_EMIT : LS_EV_SURFACE);
                        need = false;
                    }
                    if (base + __popc(m) >= n_susp_in) susp_left = false;
                }
                if (fresh_left) {
                    const unsigned m = __ballot_sync(kFullMask, need);
                    if (m) {
                        if (record && *(volatile unsigned int*)ev.count >= ev.soft_cap) {
                            fresh_left = false;  // event buffer nearly full: let the pass drain
                        } else {
                            unsigned long long base = 0;
                            if (lane_id() == __ffs(m) - 1) base = atomicAdd(rc.work_counter, (unsigned long long)__popc(m));
                            base = __shfl_sync(kFullMask, base, __ffs(m) - 1);
                            const unsigned long long item = base + rank_in_mask(m);
                            if (base + __popc(m) >= total_items) fresh_left = false;
                            if (need && item < total_items) {
                                pk.chan_run = uint32_t(div_magic(item, rc.n_pkt, rc.magic_npkt));
                                pk.pkt = rc.pkt_begin + uint32_t(item - (unsigned long long)pk.chan_run * rc.n_pkt);
                                pk.m_inter = 0; pk.nev = 0;
                                const int ctab = rc.chan_begin + int(pk.chan_run);
                                alpha_c = chan_table(ctab);
                                const uint32_t ckey = rc.chan_key0 + uint32_t(ctab);
                                const Zeta4 z = zeta_block(rc.seed, ckey, pk.pkt, 0, 0);
                                if (rc.mode == 0) {
                                    // O3: uniform point on the star-facing TOA disc, direction -s^ (or, Sect. 5.1 with
                                    // multiple scattering, the start of a transit chord, direction o^)
                                    float px, py, pz;
                                    bool dark = false;
                                    if (rc.launch_chord) {
                                        float b, X, Y, Wld;
                                        chord_point(rc, z.z0, z.z1, b, X, Y, Wld);
                                        chord_start(rc, b, X, Y, px, py, pz);
                                        dark = !(Wld > 0.f);
                                    } else {
                                        const float b = rc.geom.Rtoa * sqrtf(z.z0);
                                        float sp, cp;
                                        sincospif(2.0f * z.z1, &sp, &cp);
                                        const float h = rc.geom.Rtoa * sqrtf(1.0f - z.z0);
                                        const float ax = b * cp, ay = b * sp;
                                        px = ax * rc.e1[0] + ay * rc.e2[0] + h * rc.star[0];
                                        py = ax * rc.e1[1] + ay * rc.e2[1] + h * rc.star[1];
                                        pz = ax * rc.e1[2] + ay * rc.e2[2] + h * rc.star[2];
                                    }
                                    int j, k;
                                    locate_angles(gs, px, py, pz, j, k);
                                    pk.W = 1.0f;
                                    pk.tau_t = -logf(z.z2);
                                    pk.tau = 0.f; pk.fl_seg = 0;
                                    ray_init<DUAL>(pk.ray, gs, px, py, pz, rc.launch_dir[0], rc.launch_dir[1], rc.launch_dir[2], gs.nlev - 1,
                                             j, k, alpha_c);
                                    if (!(!DUAL && rc.forced_scatter && force_flight(rc, gs, pk.ray, alpha_c, pk.tau_t, pk.W, c_escw)))
                                        pk.tau_t *= rc.inv_stretch;
                                    st = LS_FLY;
                                    if (dark) { st = LS_IDLE; finish_packet(rc, pk); }   // chord off the stellar disc: no light to scatter
                                } else {
                                    // O4: cell ~ luminosity (Eq. 13) with composite bias xi, uniform point in the cell
                                    const int ncell = rc.geom.ncell;
                                    const double* cum = rc.Lcum + (size_t)ctab * ncell;
                                    const double Ltot = rc.Ltot[ctab];
                                    int cell;
                                    st = LS_EV_EMIT;
                                    if (!(Ltot > 0.0)) {
                                        cell = 0; st = LS_IDLE; finish_packet(rc, pk);
                                    } else if (double(z.z0) < rc.xi) {
                                        cell = min(int(floor(double(z.z0) / rc.xi * ncell)), ncell - 1);
                                    } else {
                                        const double x = (double(z.z0) - rc.xi) / (1.0 - rc.xi) * Ltot;
                                        cell = emis_search(cum, rc.Lcol + (size_t)ctab * (ncell / gs.nlev), Ltot, gs.nlev, ncell / gs.nlev, 0, ncell - 1, x);
                                    }
                                    if (st == LS_EV_EMIT) {
                                        float W = 1.0f;
                                        bool live = true;
                                        if (rc.xi > 0.0) {
                                            const double Li = rc.Lcell[(size_t)ctab * ncell + cell];
                                            live = Li > 0.0;
                                            W = live ? float(1.0 / ((1.0 - rc.xi) + rc.xi * Ltot / (double(ncell) * Li))) : 0.f;
                                        }
                                        if (!live) {
                                            st = LS_IDLE; finish_packet(rc, pk);
                                        } else {
                                            const int i = cell % gs.nlev, j = (cell / gs.nlev) % gs.nlat,
                                                      k = cell / (gs.nlev * gs.nlat);
                                            const float r = gs.R[i] * cbrtf(fmaf(z.z1, gs.qcube[i], 1.0f));
                                            const float ct = fmaf(z.z2, gs.cth[j + 1] - gs.cth[j], gs.cth[j]);
                                            const float sth = sqrtf(fmaxf(0.f, 1.0f - ct * ct));
                                            const float phi = fmaf(z.z3, gs.ph[k + 1] - gs.ph[k], gs.ph[k]);
                                            float sp, cp;
                                            sincosf(phi, &sp, &cp);
                                            pk.W = W;
                                            pk.ray.pcx = r * sth * cp; pk.ray.pcy = r * sth * sp; pk.ray.pcz = r * ct;
                                            pk.ray.u = 0.f; pk.ray.nx = 0.f; pk.ray.ny = 0.f; pk.ray.nz = 1.f;
                                            pk.ray.i = i; pk.ray.j = j; pk.ray.k = k;
                                                            }
                                    }
                                }
                            }
                        }
                    }
                }
            }
            // ---------------- events: record for the peel kernel, then absorb / scatter ----------------
            const bool is_ev = st >= LS_EV_MEDIUM && st <= LS_EV_SURFACE;
            const unsigned m_e = __ballot_sync(kFullMask, is_ev);
            if (m_e) {
                unsigned int slot = 0;
                bool have_slot = true;
                if (record) {
                    unsigned int base = 0;
                    if (lane_id() == __ffs(m_e) - 1) base = atomicAdd(ev.count, (unsigned)__popc(m_e));
                    base = __shfl_sync(kFullMask, base, __ffs(m_e) - 1);
                    slot = base + rank_in_mask(m_e);
                    have_slot = slot < ev.cap;
                }
                if (is_ev) {
                    float px, py, pz;
                    ray_position(pk.ray, px, py, pz);
                    const uint32_t cellp = pack_cell(st == LS_EV_SURFACE ? 0 : pk.ray.i, pk.ray.j, pk.ray.k);
                    const uint32_t kind = st == LS_EV_MEDIUM ? EV_MEDIUM : (st == LS_EV_EMIT ? EV_EMIT : EV_SURFACE);
                    if (!have_slot) {
                        // event buffer full: park the packet for the next pass
                        const unsigned int sidx = atomicAdd(susp_out.count, 1u);
                        if (sidx < susp_out.cap) {
                            susp_out.s0[sidx] = make_float4(px, py, pz, pk.W);
                            susp_out.s1[sidx] = make_float4(pk.ray.nx, pk.ray.ny, pk.ray.nz, __uint_as_float(cellp));
                            susp_out.s2[sidx] = make_uint4(pk.chan_run, pk.pkt, pk.m_inter, pk.nev | kind << 28);
                        } else {
                            ++c_stuck;
                        }
                        st = LS_IDLE;   // the lane goes on moving the rest of the suspended list over to the next pass
                    } else {
                        const int ctab = rc.chan_begin + int(pk.chan_run);
                        const uint32_t ckey = rc.chan_key0 + uint32_t(ctab);
                        const int cell = (pk.ray.k * gs.nlat + pk.ray.j) * gs.nlev + pk.ray.i;
                        const uint32_t meta = kind | batch_of(rc, pk.pkt) << 2 | pk.chan_run << 8;
                        ++c_events;
                        ++pk.nev;
                        if (st == LS_EV_MEDIUM) {
                            const float4 pr = __ldg(rc.prop + (size_t)ctab * rc.geom.ncell + cell);
                            if (record) {
                                write_event(ev, slot, px, py, pz, pk.W, pk.ray.nx, pk.ray.ny, pk.ray.nz, pk.m_inter, cellp,
                                            meta, pk.pkt, pr);
                            }
                            ++pk.m_inter;
                            const Zeta4 z = zeta_block(rc.seed, ckey, pk.pkt, pk.m_inter, 1);
                            float ct = 0.f;
                            if ((rc.max_events && int(pk.m_inter) == rc.max_events) || !rc.scatter_on ||
                                !medium_interaction(rc, pr, z, ckey, pk.pkt, pk.m_inter, pk.W, ct)) {
                                ++c_abs; st = LS_IDLE; finish_packet(rc, pk);       // L192: absorbed
                            } else {
                                float nx = pk.ray.nx, ny = pk.ray.ny, nz = pk.ray.nz;
                                rotate_dir(nx, ny, nz, ct, z.z2);
                                pk.tau_t = -logf(z.z3); pk.tau = 0.f; pk.fl_seg = 0;
                                ray_init<DUAL>(pk.ray, gs, px, py, pz, nx, ny, nz, pk.ray.i, pk.ray.j, pk.ray.k, alpha_c);
                                if (!(!DUAL && rc.forced_scatter == 2 && force_flight(rc, gs, pk.ray, alpha_c, pk.tau_t, pk.W, c_escw)))
                                    pk.tau_t *= rc.inv_stretch;
                                st = LS_FLY;
                            }
                        } else if (st == LS_EV_EMIT) {
                            if (record) {
                                write_event(ev, slot, px, py, pz, pk.W, 0.f, 0.f, 1.f, pk.m_inter, cellp, meta, pk.pkt,
                                            make_float4(0.f, 0.f, 0.f, 0.f));
                            }
                            if (!rc.scatter_on) {
                                ++c_abs; st = LS_IDLE; finish_packet(rc, pk);
                            } else {
                                const Zeta4 z = zeta_block(rc.seed, ckey, pk.pkt, 1, 0);
                                const float nz = fmaf(2.0f, z.z0, -1.0f);   // Eq. 2
                                const float ns = sqrtf(fmaxf(0.f, 1.0f - nz * nz));
                                float sp, cp;
                                sincospif(2.0f * z.z1, &sp, &cp);
                                pk.tau_t = -logf(z.z2); pk.tau = 0.f; pk.fl_seg = 0;
                                ray_init<DUAL>(pk.ray, gs, px, py, pz, ns * cp, ns * sp, nz, pk.ray.i, pk.ray.j, pk.ray.k, alpha_c);
                                if (!(!DUAL && rc.forced_scatter == 2 && force_flight(rc, gs, pk.ray, alpha_c, pk.tau_t, pk.W, c_escw)))
                                    pk.tau_t *= rc.inv_stretch;
                                st = LS_FLY;
                            }
                        } else {  // Lambert surface (O7, Eq. 3-4)
                            const float a = rc.surface_albedo;
                            const float rn = rsqrtf(fmaf(px, px, fmaf(py, py, pz * pz)));
                            float hx = px * rn, hy = py * rn, hz = pz * rn;
                            if (record) {
                                write_event(ev, slot, px, py, pz, pk.W, hx, hy, hz, pk.m_inter, cellp, meta, pk.pkt,
                                            make_float4(0.f, 0.f, 0.f, 0.f));
                            }
                            ++pk.m_inter;
                            const Zeta4 z = zeta_block(rc.seed, ckey, pk.pkt, pk.m_inter, 3);
                            if (rc.max_events && int(pk.m_inter) == rc.max_events) {
                                ++c_abs; st = LS_IDLE; finish_packet(rc, pk);
                            } else if (z.z0 >= a) {
                                ++c_surf; st = LS_IDLE; finish_packet(rc, pk);
                            } else {
                                rotate_dir(hx, hy, hz, sqrtf(z.z1), z.z2);      // Eq. 4 about the normal
                                pk.tau_t = -logf(z.z3); pk.tau = 0.f; pk.fl_seg = 0;
                                ray_init<DUAL>(pk.ray, gs, px, py, pz, hx, hy, hz, 0, pk.ray.j, pk.ray.k, alpha_c);
                                if (!(!DUAL && rc.forced_scatter == 2 && force_flight(rc, gs, pk.ray, alpha_c, pk.tau_t, pk.W, c_escw)))
                                    pk.tau_t *= rc.inv_stretch;
                                st = LS_FLY;
                            }
                        }
                    }
                }
            }
        }
        // ---------------- lateral crossings: cone / half-plane root updates, batched across the warp ----------------
        if (m_park && (__popc(m_park) >= rc.t_lateral || starving)) {
            if (st == LS_PARK) {
                ray_lateral<DUAL>(pk.ray, gs, alpha_c);
                st = LS_FLY;
            }
        }
        if (__ballot_sync(kFullMask, st == LS_FLY) == 0) {
            if (__ballot_sync(kFullMask, st != LS_DONE) == 0) break;
            continue;
        }
        // ---------------- march: up to KSTEPS radial cell crossings per lane ----------------
#pragma unroll
        for (int s = 0; s < KSTEPS; ++s) {
            if (st == LS_FLY) {
                const int rs = ray_step<DUAL>(pk.ray, gs, pk.tau, pk.tau_t, &pk.tau_b);
                ++c_seg32;
                if (DUAL && rs != RAY_FLYING && rs != RAY_PARK) {   // the flight is over: Eq. 12
                    pk.W *= expf(-pk.tau_b);
                    pk.tau_b = 0.f;
                }
                if (!DUAL && rs != RAY_FLYING && rs != RAY_PARK) pk.W *= stretch_weight(rc, rs, pk.tau);
                if (rs == RAY_FLYING) {
                    if (++pk.fl_seg > rc.geom.maxseg) st = LS_END_STUCK;
                } else if (rs == RAY_PARK) {
                    st = (++pk.fl_seg > rc.geom.maxseg) ? LS_END_STUCK : LS_PARK;
                } else if (rs == RAY_LIMIT) {
                    st = LS_EV_MEDIUM;
                } else if (rs == RAY_ESCAPE) {
                    st = LS_END_ESC;
                } else {  // RAY_SURFACE
                    st = rc.surface_albedo > 0.f ? LS_EV_SURFACE : LS_END_SURF;
                }
            }
        }
    }

    // counters: warp reduce, one atomic per warp
    c_seg += c_seg32;
    c_events = warp_sum_u64(c_events); c_seg = warp_sum_u64(c_seg); c_esc = warp_sum_u64(c_esc);
    c_abs = warp_sum_u64(c_abs); c_surf = warp_sum_u64(c_surf); c_stuck = warp_sum_u64(c_stuck);
    c_escw = warp_sum_f64(c_escw);
    if (lane_id() == 0) {
        if (c_events) atomicAdd(&rc.counters->events, c_events);
        if (c_seg) atomicAdd(&rc.counters->seg_transport, c_seg);
        if (c_esc) atomicAdd(&rc.counters->escaped, c_esc);
        if (c_abs) atomicAdd(&rc.counters->absorbed, c_abs);
        if (c_surf) atomicAdd(&rc.counters->surface, c_surf);
        if (c_stuck) atomicAdd(&rc.counters->stuck, c_stuck);
        if (c_escw != 0.0) atomicAdd(&rc.counters->escaped_weight, c_escw);
    }
}

}  // namespace gcmcrt
#include "wavefront.cuh"
namespace gcmcrt {

// ---------------------------------------------------------------------------------------------------------
// Peel-off kernel (A7 + A9).  Events arrive sorted by (channel, cell) (sort.cuh): a warp takes 32 consecutive
// events, one per lane, and integrates their rays toward one observer at a time -- 32 parallel rays that start in
// the same or neighbouring cells, so the lanes read the same extinction sectors, cross the same shells in the same
// step and finish within a few steps of each other.  Cone / half-plane crossings are batched across the warp
// (ray_lateral).  f = pref * Theta * exp(-tau_obs) (Eq. 14) goes to warp-private shared-memory bins [obs][batch]
// of the warp's current channel, flushed to the fp64 global sums when the channel changes and at the end.
// ---------------------------------------------------------------------------------------------------------
__device__ __forceinline__ void peel_flush_bins(const RunConst& rc, float* bins, int nbins, int warp_chan)
{
    for (int t = lane_id(); t < nbins; t += 32) {
        const float v = bins[t];
        if (v != 0.f) {
            const int o = t / rc.n_batches, bt = t - o * rc.n_batches;
            atomicAdd(rc.flux + ((size_t)warp_chan * rc.n_obs_total + rc.obs_first + o) * rc.n_batches + bt, double(v));
            bins[t] = 0.f;
        }
    }
}

constexpr int kPeelChunk = 128;   // consecutive sorted events a warp takes per atomic (4 rounds of 32)

template <int KSTEPS, bool HORIZON>
__global__ void __launch_bounds__(kPeelThreads, 4)
peel_kernel(const __grid_constant__ RunConst rc, const EventBuf ev, const unsigned int* __restrict__ perm)
{
    extern __shared__ float smem_f[];
    const GeomSmem gs = load_geom(rc.geom, smem_f);
    const int nbins = rc.n_obs_run * rc.n_batches;
    float* bins = smem_f + ((rc.geom.tab_floats + 31) & ~31) + (threadIdx.x >> 5) * nbins;
    for (int t = lane_id(); t < nbins; t += 32) bins[t] = 0.f;
    __syncthreads();

    const unsigned int n_events = min(*ev.count, ev.cap);
    int warp_chan = -1;  // channel (run-local) the warp's bins belong to
    unsigned long long c_seg = 0, c_rays = 0;

    for (;;) {
        unsigned long long base = 0;
        if (lane_id() == 0) base = atomicAdd(rc.ray_counter, (unsigned long long)kPeelChunk);
        base = __shfl_sync(kFullMask, base, 0);
        if (base >= n_events) break;
        const unsigned int chunk_end = (unsigned int)min((unsigned long long)n_events, base + kPeelChunk);
        unsigned int slot_next = 0;   // record of this lane's event in the next round of 32
        if ((unsigned int)base + lane_id() < chunk_end) slot_next = __ldg(perm + (unsigned int)base + lane_id());
        for (unsigned int r0 = (unsigned int)base; r0 < chunk_end; r0 += 32) {
            const unsigned int rank = r0 + lane_id();
            const bool have = rank < chunk_end;
            float4 a = make_float4(0.f, 0.f, 0.f, 0.f), b = a, c = a, pr = a;
            if (have) {
                GCMCRT_CHECK(slot_next < n_events);
                const float4* r = ev.rec + 4 * (size_t)slot_next;
                a = __ldg(r); b = __ldg(r + 1); c = __ldg(r + 2); pr = __ldg(r + 3);
            }
            if (rank + 32 < chunk_end) {   // next round's records on their way while this round's rays are integrated
                slot_next = __ldg(perm + rank + 32);
                asm volatile("prefetch.global.L1 [%0];" ::"l"(ev.rec + 4 * (size_t)slot_next));
            }
            const uint32_t meta = __float_as_uint(c.z);
            const uint32_t kind = meta & 3u;
            const int chan = have ? int(meta >> 8) : -1;
            const int bt = int((meta >> 2) & 63u);
            int ci, cj, ck;
            unpack_cell(__float_as_uint(c.y), ci, cj, ck);
            GCMCRT_CHECK(!have || (chan >= 0 && chan < rc.n_chan_run && bt < rc.n_batches && ci < gs.nlev && cj < gs.nlat && ck < gs.nlon));
            const float* alpha_c = rc.alpha + (size_t)(rc.chan_begin + max(chan, 0)) * rc.geom.alpha_stride;
            // what the event scatters toward an observer: W omega (medium, Eq. 14), W (emission), W a (surface)
            float wsca = a.w, pgas = 0.f, g = 0.f;
            if (rc.launch_chord && have)   // scattered light of a transit chord: -W_ld b dOmega of the packet's chord (N12)
                wsca *= -chord_scale(rc, rc.chan_key0 + uint32_t(rc.chan_begin + chan), __float_as_uint(c.w));
            if (have && kind == EV_MEDIUM) {
                wsca *= pr.x; pgas = pr.y; g = pr.z;
            } else if (kind == EV_SURFACE) {
                wsca *= rc.surface_albedo;
            }
            // the warp's bins follow the newest channel; stragglers of older channels go straight to global memory
            int mx = chan;
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) mx = max(mx, __shfl_xor_sync(kFullMask, mx, o));
            if (mx > warp_chan) {
                if (warp_chan >= 0) {
                    __syncwarp();
                    peel_flush_bins(rc, bins, nbins, warp_chan);
                    __syncwarp();
                }
                warp_chan = mx;
            }
            for (int obs = 0; obs < rc.n_obs_run; ++obs) {
                const float* od = rc.obs[rc.obs_first + obs];
                const float ox = od[0], oy = od[1], oz = od[2];
                const float mu = b.x * ox + b.y * oy + b.z * oz;
                float theta;
                if (kind == EV_MEDIUM) {  // C6: mixture phase function, per steradian (Eq. 5, Eq. 7)
                    const float hg = phase_cloud(rc.cloud_phase, g, mu);
                    const float ray_p = (3.0f / (16.0f * kPi)) * fmaf(mu, mu, 1.0f);
                    theta = pgas * ray_p + (1.0f - pgas) * hg;
                } else if (kind == EV_EMIT) {
                    theta = 1.0f / (4.0f * kPi);
                } else {
                    theta = fmaxf(mu, 0.0f) / kPi;
                }
                const float pref = wsca * theta;
                Ray ray{};
                float tau = 0.f;
                int st = RAY_NONE;      // lane state = ray status: RAY_FLYING marches, RAY_PARK waits for ray_lateral
                unsigned int seg32 = 0;
                // a ray that descends and does not turn inside the grid ends on the lower boundary: nothing of it reaches
                // the observer (Eq. 14 along a ray that leaves through the top), so it is not marched at all -- with
                // observers all around the orbit these are the long rays through the deep atmosphere.  Most of them point
                // well below the horizon of the lower boundary (impact parameter d < R_0 by more than any rounding of this
                // fp32 estimate: r^2 ~ 1e16 m^2 carries ~1e9, the margin is 1e-4 R_0^2); the lanes of a warp share a cell and
                // an observer, so a warp of such rays does not even set them up.  Every other ray is decided by the march's
                // own double-float expression.
                const bool go = have && pref > 0.0f;
                bool below = false;
                if (HORIZON) {
                    const float b0 = fmaf(a.x, ox, fmaf(a.y, oy, a.z * oz));
                    const float dq = fmaf(-b0, b0, fmaf(a.x, a.x, fmaf(a.y, a.y, a.z * a.z)));
                    below = b0 < 0.0f && dq < rc.geom.R0 * rc.geom.R0 * (1.0f - 1e-4f);
                }
                if (go) { ++c_rays; st = RAY_SURFACE; }
                if (!HORIZON || __any_sync(kFullMask, go && !below)) {
                    if (go) {
                        ray_init(ray, gs, a.x, a.y, a.z, ox, oy, oz, ci, cj, ck, alpha_c);
                        st = (ray.rad_step < 0 && ray.i_turn < 0) ? RAY_SURFACE : RAY_FLYING;
                    }
                }
                // all lanes start together, so one warp-uniform step budget guards against a ray that never ends
                for (int it = 0; it <= rc.geom.maxseg; it += KSTEPS) {
                    const unsigned m_fly = __ballot_sync(kFullMask, st == RAY_FLYING);
                    const unsigned m_park = __ballot_sync(kFullMask, st == RAY_PARK);
                    if ((m_fly | m_park) == 0) break;
                    if (m_park && (__popc(m_park) >= rc.t_lateral || m_fly == 0)) {
                        if (st == RAY_PARK) {
                            ray_lateral(ray, gs, alpha_c);
                            st = RAY_FLYING;
                        }
                    }
                    if (st == RAY_FLYING) st = ray_run<KSTEPS>(ray, gs, tau, rc.tau_cut, seg32);   // lanes in flight step together
                }
                c_seg += seg32;
                // ---------------- rays that reached the top of the atmosphere: Eq. 14 ----------------
                if (st == RAY_ESCAPE) {
                    const float f = rc.launch_chord ? -pref * expf(-tau) : pref * expf(-tau);
                    if (chan == warp_chan) atomicAdd(bins + obs * rc.n_batches + bt, f);
                    else atomicAdd(rc.flux + ((size_t)chan * rc.n_obs_total + rc.obs_first + obs) * rc.n_batches + bt, double(f));
                    if (rc.image) {
                        const int o = rc.obs_first + obs;
                        const float X = a.x * rc.img_ex[o][0] + a.y * rc.img_ex[o][1] + a.z * rc.img_ex[o][2];
                        const float Y = a.x * rc.img_ey[o][0] + a.y * rc.img_ey[o][1] + a.z * rc.img_ey[o][2];
                        const int ix = min(max(int(floorf((X / rc.geom.Rtoa + 1.0f) * 0.5f * rc.npix)), 0), rc.npix - 1);
                        const int iy = min(max(int(floorf((Y / rc.geom.Rtoa + 1.0f) * 0.5f * rc.npix)), 0), rc.npix - 1);
                        atomicAdd(rc.image + ((size_t)chan * rc.n_obs_total + o) * rc.npix * rc.npix + iy * rc.npix + ix, f);
                    }
                }
                if (rc.contrib) {
                    // Sect. 6, Eq. 32: f per event cell, thermal and scattered apart.  The lanes are sorted by
                    // (channel, cell group), so the lanes of one cell are mostly neighbours: sum each RUN of consecutive
                    // lanes with the same (channel, cell) with a segmented shuffle reduction (both components at once) and
                    // let the run's first lane do the atomics.  A merge never reaches across a run boundary, so a cell
                    // whose lanes are not contiguous (coarse sort keys, channels folded into one bin) is simply several runs.
                    const unsigned ckey = have ? unsigned((ck * gs.nlat + cj) * gs.nlev + ci) : 0xffffffffu;
                    const float f = st == RAY_ESCAPE ? pref * expf(-tau) : 0.f;
                    float v0 = kind == EV_EMIT ? f : 0.f, v1 = kind == EV_EMIT ? 0.f : f;
                    const unsigned kp = __shfl_up_sync(kFullMask, ckey, 1);
                    const int cp = __shfl_up_sync(kFullMask, chan, 1);
                    const unsigned heads = __ballot_sync(kFullMask, lane_id() == 0 || kp != ckey || cp != chan);
                    const unsigned after = lane_id() < 31 ? heads >> (lane_id() + 1) : 0u;
                    const int run_end = after ? lane_id() + __ffs(after) : 32;   // first lane of the next run
#pragma unroll
                    for (int off = 1; off < 32; off <<= 1) {
                        const float w0 = __shfl_down_sync(kFullMask, v0, off), w1 = __shfl_down_sync(kFullMask, v1, off);
                        if (lane_id() + off < run_end) { v0 += w0; v1 += w1; }
                    }
                    if (have && ((heads >> lane_id()) & 1u)) {
                        float* dst = rc.contrib + ((size_t)chan * rc.n_obs_total + rc.obs_first + obs) * 2 * rc.geom.ncell + ckey;
                        if (v0 != 0.f) atomicAdd(dst, v0);
                        if (v1 != 0.f) atomicAdd(dst + rc.geom.ncell, v1);
                    }
                }
                __syncwarp();
            }
        }
    }
    __syncwarp();
    if (warp_chan >= 0) peel_flush_bins(rc, bins, nbins, warp_chan);
    c_seg = warp_sum_u64(c_seg); c_rays = warp_sum_u64(c_rays);
    if (lane_id() == 0) {
        if (c_seg) atomicAdd(&rc.counters->seg_peel, c_seg);
        if (c_rays) atomicAdd(&rc.counters->rays_peel, c_rays);
    }
}

// ---------------------------------------------------------------------------------------------------------
// Transmission (Sect. 5.1, Eq. 20-23): one random transit chord per packet, toward observer `o`.
// ---------------------------------------------------------------------------------------------------------
struct TransParams {
    int o;                   // observer index (row of rc.obs, column of flux)
    float ex[3], ey[3];      // sky-plane frame of the observer (C19)
    float star_radius, planet_x, planet_y, ld_c1, ld_c2;
};

template <int KSTEPS>
__global__ void __launch_bounds__(256, 3)
transmission_kernel(const __grid_constant__ RunConst rc, const TransParams tp, const unsigned long long total_items)
{
    extern __shared__ float smem_f[];
    const GeomSmem gs = load_geom(rc.geom, smem_f);
    __syncthreads();
    const float ox = rc.obs[tp.o][0], oy = rc.obs[tp.o][1], oz = rc.obs[tp.o][2];
    const float R0 = rc.geom.R0, Rt = rc.geom.Rtoa;
    unsigned long long c_seg = 0, c_ev = 0, c_stuck = 0;
    const unsigned long long stride = (unsigned long long)gridDim.x * blockDim.x;
    for (unsigned long long base = ((unsigned long long)blockIdx.x * blockDim.x + threadIdx.x) & ~31ull; base < total_items;
         base += stride) {
        const unsigned long long item = base + lane_id();
        const bool active = item < total_items;
        uint32_t chan_run = 0, pkt = 0;
        Ray ray{};
        float b = 0.f, W = 0.f, tau = 0.f;
        int st = RAY_NONE;
        const float* alpha_c = rc.alpha;
        if (active) {
            chan_run = uint32_t(div_magic(item, rc.n_pkt, rc.magic_npkt));
            pkt = rc.pkt_begin + uint32_t(item - (unsigned long long)chan_run * rc.n_pkt);
            const int ctab = rc.chan_begin + int(chan_run);
            alpha_c = rc.alpha + (size_t)ctab * rc.geom.alpha_stride;
            const Zeta4 z = zeta_block(rc.seed, rc.chan_key0 + uint32_t(ctab), pkt, 0, 0);
            b = fmaf(z.z0, Rt - R0, R0);                       // uniform in b: Eq. 21 carries the factor b_i
            float sp, cp;
            sincospif(2.0f * z.z1, &sp, &cp);
            const float X = b * cp, Y = b * sp, h = sqrtf(fmaxf(0.f, (Rt - b) * (Rt + b)));
            const float px = X * tp.ex[0] + Y * tp.ey[0] - h * ox;
            const float py = X * tp.ex[1] + Y * tp.ey[1] - h * oy;
            const float pz = X * tp.ex[2] + Y * tp.ey[2] - h * oz;
            W = 1.0f;
            if (tp.star_radius > 0.f) {                         // Eq. 22-23
                const float sx = (tp.planet_x + X) / tp.star_radius, sy = (tp.planet_y + Y) / tp.star_radius;
                const float rho2 = fmaf(sx, sx, sy * sy);
                const float mu1 = 1.0f - sqrtf(fmaxf(0.f, 1.0f - rho2));
                W = rho2 >= 1.0f ? 0.f : 1.0f - tp.ld_c1 * mu1 - tp.ld_c2 * mu1 * mu1;
            }
            int j, k;
            locate_angles(gs, px, py, pz, j, k);
            ray_init(ray, gs, px, py, pz, ox, oy, oz, gs.nlev - 1, j, k, alpha_c);
            st = RAY_FLYING;
            ++c_ev;
        }
        unsigned int seg32 = 0;
        for (int it = 0; it <= rc.geom.maxseg; it += KSTEPS) {
            const unsigned m_fly = __ballot_sync(kFullMask, st == RAY_FLYING);
            const unsigned m_park = __ballot_sync(kFullMask, st == RAY_PARK);
            if ((m_fly | m_park) == 0) break;
            if (m_park && (__popc(m_park) >= rc.t_lateral || m_fly == 0)) {
                if (st == RAY_PARK) { ray_lateral(ray, gs, alpha_c); st = RAY_FLYING; }
            }
            if (st == RAY_FLYING) st = ray_run<KSTEPS>(ray, gs, tau, rc.tau_cut, seg32);   // beyond tau_cut the chord is opaque: 1 - e^-tau = 1
        }
        c_seg += seg32;
        float v = 0.f;
        if (active) {
            if (st == RAY_ESCAPE) v = W * b * -expm1f(-tau);
            else if (st == RAY_LIMIT || st == RAY_SURFACE) v = W * b;
            else ++c_stuck;
        }
        // items of a warp are consecutive packets: (channel, batch) runs are contiguous -> segmented reduction
        const int key = active ? int(chan_run) * rc.n_batches + int(batch_of(rc, pkt)) : -1;
        double dv = double(v);
#pragma unroll
        for (int off = 1; off < 32; off <<= 1) {
            const double w = __shfl_down_sync(kFullMask, dv, off);
            const int kk = __shfl_down_sync(kFullMask, key, off);
            if (lane_id() + off < 32 && kk == key) dv += w;
        }
        const int kp = __shfl_up_sync(kFullMask, key, 1);
        if (active && (lane_id() == 0 || kp != key) && dv != 0.0) {
            const int bt = key - int(chan_run) * rc.n_batches;
            atomicAdd(rc.flux + ((size_t)chan_run * rc.n_obs_total + tp.o) * rc.n_batches + bt, dv);
        }
    }
    c_seg = warp_sum_u64(c_seg); c_ev = warp_sum_u64(c_ev); c_stuck = warp_sum_u64(c_stuck);
    if (lane_id() == 0) {
        if (c_seg) atomicAdd(&rc.counters->seg_peel, c_seg);
        if (c_ev) { atomicAdd(&rc.counters->events, c_ev); atomicAdd(&rc.counters->rays_peel, c_ev); }
        if (c_stuck) atomicAdd(&rc.counters->stuck, c_stuck);
    }
}

// ---------------------------------------------------------------------------------------------------------
// A10: value and batch-means sigma (C12) per (channel, observer).
// ---------------------------------------------------------------------------------------------------------
__global__ void normalise_kernel(int n_chan_run, int n_obs, int n_batches, unsigned long long N, unsigned long long lo,
                                 unsigned long long hi, const double* __restrict__ flux, const double* __restrict__ Ltot,
                                 int emission, double scale_const, double* __restrict__ value, double* __restrict__ sigma)
{
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= n_chan_run * n_obs) return;
    const double* S = flux + (size_t)t * n_batches;
    double sum = 0.0, n_run = 0.0, m1 = 0.0, m2 = 0.0;
    int used = 0;
    for (int b = 0; b < n_batches; ++b) {
        unsigned long long e0 = ((unsigned long long)b * N + n_batches - 1) / n_batches;
        unsigned long long e1 = ((unsigned long long)(b + 1) * N + n_batches - 1) / n_batches;
        e0 = e0 < lo ? lo : e0;
        e1 = e1 > hi ? hi : e1;
        const double cnt = e1 > e0 ? double(e1 - e0) : 0.0;
        sum += S[b];
        n_run += cnt;
        if (cnt > 0.0) { const double bm = S[b] / cnt; m1 += bm; m2 += bm * bm; ++used; }
    }
    double mean = n_run > 0.0 ? sum / n_run : 0.0;
    double sg = 0.0;
    if (used > 1) {
        const double mu = m1 / used;
        const double var = fmax(0.0, (m2 - used * mu * mu) / (used - 1));
        sg = sqrt(var / used);
    }
    const double scale = emission == 1 ? Ltot[t] : (emission == 2 ? scale_const : 1.0);   // Eq. 28 | Eq. 21 | Eq. 24
    if (value) value[t] = mean * scale;
    if (sigma) sigma[t] = sg * scale;
}

// ---------------------------------------------------------------------------------------------------------
// Test-only kernels.
// ---------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(128) debug_ray_tau_kernel(const GeomParams g, const float* __restrict__ alpha_c, long n,
                                                           const float* __restrict__ pos, const float* __restrict__ dir,
                                                           float* __restrict__ tau_out, int* __restrict__ hit)
{
    extern __shared__ float smem_f[];
    const GeomSmem gs = load_geom(g, smem_f);
    __syncthreads();
    const long m = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (m >= n) return;
    const float px = pos[3 * m], py = pos[3 * m + 1], pz = pos[3 * m + 2];
    int j, k;
    locate_angles(gs, px, py, pz, j, k);
    const int i = locate_ascending(gs.R, gs.nlev, sqrtf(px * px + py * py + pz * pz));
    Ray ray{};
    ray_init(ray, gs, px, py, pz, dir[3 * m], dir[3 * m + 1], dir[3 * m + 2], i, j, k, alpha_c);
    float tau = 0.f;
    int rs = RAY_FLYING, nseg = 0;
    while (rs == RAY_FLYING && nseg++ <= g.maxseg) {
        rs = ray_step(ray, gs, tau, kInf);
        if (rs == RAY_PARK) { ray_lateral(ray, gs, alpha_c); rs = RAY_FLYING; }
    }
    tau_out[m] = tau;
    if (hit) hit[m] = rs == RAY_SURFACE ? 1 : (rs == RAY_ESCAPE ? 0 : -1);
}

__global__ void debug_philox_kernel(long n, const uint32_t* __restrict__ ctr, const uint32_t* __restrict__ key,
                                    uint32_t* __restrict__ out)
{
    const long m = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (m >= n) return;
    const Philox4 r = philox4x32_10(ctr[4 * m], ctr[4 * m + 1], ctr[4 * m + 2], ctr[4 * m + 3], key[2 * m], key[2 * m + 1]);
    out[4 * m] = r.x; out[4 * m + 1] = r.y; out[4 * m + 2] = r.z; out[4 * m + 3] = r.w;
}

}  // namespace gcmcrt

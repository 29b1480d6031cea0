// ray.cuh -- fp32 ray marcher through the spherical-polar grid (A6 / A7), shared by the transport kernel and
// the peel-off ray integrator.
//
// Formulation (differs from the paper-era "recompute six face distances from the current position" scheme the
// oracle follows): a ray is described once by its invariants -- closest-approach point pc = p0 - n (p0.n), direction
// n, impact parameter d^2 = |p0 x n|^2 -- and a running signed distance u from the closest-approach point, so that
//   r(u)^2 = d^2 + u^2,   p(u) = pc + n u.
// Every face crossing is then a closed-form root in u that depends only on the invariants and the face:
//   shell R_k:           u = -/+ sqrt(R_k^2 - d^2)                      (1 MUFU)
//   cone cos(theta)=c:   (n_z^2-c^2) u^2 + 2 z_c n_z u + (z_c^2 - c^2 d^2) = 0
//   half-plane phi_e:    u = -(pc.N)/(n.N),  N = (-sin phi_e, cos phi_e, 0)
// Only the face family that was just crossed is recomputed, positions are never advanced incrementally (no drift),
// cell indices are tracked by crossings (never re-located from coordinates), and the face just crossed is excluded
// by the strict comparison root > u, which is exact because the recomputed root is bit-identical to the u it set.
//
// The march is split in two: ray_step() is the radial fast path (shell crossings: ~30 instructions, no global
// address arithmetic beyond one IMAD.WIDE, the extinction of the next cell prefetched one step ahead); a cone or
// half-plane crossing stops it with RAY_PARK and is completed by ray_lateral(), which the kernels batch across the
// warp.  The staged extinction table has one guard entry below and above every column so that the prefetch needs
// no clamping.
#pragma once
#include "device_common.cuh"

namespace gcmcrt {

// Padded column length of the staged extinction table: nlev + 2 guard entries, rounded up to whole 32 B sectors.
__host__ __device__ inline int alpha_col_stride(int nlev) { return (nlev + 2 + 7) & ~7; }

// Geometry tables, staged by the host into one device array and copied to shared memory by every CTA.
struct GeomParams {
    int nlev, nlat, nlon, ncell;
    const float* tab;  // packed: R2pair[2(nlev+1)] R[nlev+1] qcube[nlev] cth[nlat+1] cph[nlon+1] sph[nlon+1] ph[nlon+1]
    int tab_floats;
    float Rtoa, R0;
    int maxseg;
    int col_stride;    // alpha_col_stride(nlev)
    long long alpha_stride;  // floats per channel of the staged extinction table: nlat * nlon * col_stride
};

struct GeomSmem {
    uint32_t r2_saddr; // shared-space address of R2: the shell roots load it with one LDS.64 and no generic-address set-up
    const float2* R2;  // (high, low) parts of R_k^2
    const float *R, *qcube, *cth, *cph, *sph, *ph;
    int nlev, nlat, nlon, col_stride;
};

__device__ __forceinline__ GeomSmem load_geom(const GeomParams& g, float* smem)
{
    for (int t = threadIdx.x; t < g.tab_floats; t += blockDim.x) smem[t] = g.tab[t];
    GeomSmem s;
    s.nlev = g.nlev; s.nlat = g.nlat; s.nlon = g.nlon; s.col_stride = g.col_stride;
    s.R2 = reinterpret_cast<const float2*>(smem);
    s.r2_saddr = static_cast<uint32_t>(__cvta_generic_to_shared(smem));
    s.R = smem + 2 * (g.nlev + 1);
    s.qcube = s.R + (g.nlev + 1);
    s.cth = s.qcube + g.nlev;
    s.cph = s.cth + (g.nlat + 1);
    s.sph = s.cph + (g.nlon + 1);
    s.ph = s.sph + (g.nlon + 1);
    return s;
}

// Ray status doubles as the lane state of the kernels: RAY_FLYING lanes march, RAY_PARK lanes wait for
// ray_lateral(), everything else is a finished flight.
enum RayStatus : int { RAY_FLYING = 0, RAY_LIMIT = 1, RAY_ESCAPE = 2, RAY_SURFACE = 3, RAY_STUCK = 4, RAY_PARK = 5,
                       RAY_NONE = 6 };

struct Ray {
    float pcx, pcy, pcz;  // closest-approach point
    float nx, ny, nz;     // unit direction
    float d2;             // impact parameter squared: high part of the double-float (d2, d2lo)
    float d2lo;           // low part: R_k^2 - d^2 cancels catastrophically in plain fp32 for grazing rays
    float u;              // signed distance from the closest-approach point
    float u_rad, u_lat, u_lon;  // next crossing of each face family
    float alpha;          // extinction of the current cell
    float alpha_n;        // prefetched extinction of the radial neighbour (i + rad_step) in the same column
    float beta, beta_n;   // DUAL marches only (continuous absorption, Eq. 12): the second extinction of the same cells
    const float* pn;      // address of the extinction prefetched next, in the column of (j, k): column + i + rad_step
                          // (every column has a guard entry below level 0 and above level nlev - 1)
    int i, j, k;          // cell
    int ish;              // index of the shell the ray crosses next: i while moving inward, i + 1 outward
    int i_turn;           // cell in which an inward ray turns outward (its inner shell lies inside the impact
                          // parameter); below every cell index when the ray never turns inside the grid
    int rad_step, lat_step, lon_step;
};

__device__ __forceinline__ float shell_q(const Ray& r, const GeomSmem& s, int idx)
{
    float hi, lo;
    asm("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(hi), "=f"(lo) : "r"(s.r2_saddr + 8u * uint32_t(idx)));
    return (hi - r.d2) + (lo - r.d2lo);
}

// Next shell crossing at the start of a ray, and where an inward ray will turn.
__device__ __forceinline__ void ray_setup_rad(Ray& r, const GeomSmem& s)
{
    r.i_turn = -2;
    if (r.u < 0.0f) {  // inward phase: the inner shell is hit iff it lies outside the impact parameter
        const float q = shell_q(r, s, r.i);
        if (q > 0.0f) {
            r.u_rad = -sqrt_approx(q);
            r.rad_step = -1;
            r.ish = r.i;
            // innermost shell the ray reaches = smallest k in [0, i] with R_k^2 - d^2 > 0 (same double-float
            // expression as every shell root, so the march never asks for a shell it decided it cannot reach);
            // the ray turns in the cell below it (k = 0: it reaches the lower boundary instead)
            int lo = 0, hi = r.i;   // invariant: shell hi is reached
            while (lo < hi) {
                const int mid = (lo + hi) >> 1;
                if (shell_q(r, s, mid) > 0.0f) hi = mid; else lo = mid + 1;
            }
            r.i_turn = hi - 1;
            return;
        }
    }
    r.u_rad = sqrt_approx(fmaxf(shell_q(r, s, r.i + 1), 0.0f));
    r.rad_step = 1;
    r.ish = r.i + 1;
}

__device__ __forceinline__ void ray_cone_roots(const Ray& r, float c, int step, float& best, int& best_step)
{
    if (fabsf(c) < 1e-6f) {  // theta = pi/2: the plane z = 0
        const float ur = -r.pcz * rcp_approx(r.nz);
        if (ur > r.u && ur < best) { best = ur; best_step = step; }
        return;
    }
    const float c2 = c * c;
    const float A = fmaf(r.nz, r.nz, -c2);
    const float B = r.pcz * r.nz;
    const float C = fmaf(r.pcz, r.pcz, -c2 * r.d2);
    const float inner = fmaf(r.d2, A, r.pcz * r.pcz);  // disc = c^2 (z_c^2 + d^2 A)
    if (!(inner >= 0.0f)) return;
    const float sq = fabsf(c) * sqrt_approx(inner);
    const float q = -(B + copysignf(sq, B));
    const float u1 = q * rcp_approx(A);   // A == 0 -> inf / nan: rejected by the comparisons below
    const float u2 = C * rcp_approx(q);
    if (u1 > r.u && u1 < best && fmaf(r.nz, u1, r.pcz) * c > 0.0f) { best = u1; best_step = step; }
    if (u2 > r.u && u2 < best && fmaf(r.nz, u2, r.pcz) * c > 0.0f) { best = u2; best_step = step; }
}

__device__ __forceinline__ void ray_setup_lat(Ray& r, const GeomSmem& s)
{
    float best = kInf;
    int step = 0;
    if (s.nlat > 1) {
        // d cos(theta) / du has the sign of n_z d^2 - z_c u, which changes at most once along a line: the ray can
        // only reach the cone it is moving toward unless it turns first, so the other cone is asked only when the
        // first has no crossing ahead (pole edges are no surfaces)
        const bool up = fmaf(r.nz, r.d2, -r.pcz * r.u) > 0.0f;   // colatitude decreasing
        const int e1 = up ? r.j : r.j + 1, s1 = up ? -1 : 1;
        if (e1 > 0 && e1 < s.nlat) ray_cone_roots(r, s.cth[e1], s1, best, step);
        if (step == 0) {
            const int e2 = up ? r.j + 1 : r.j;
            if (e2 > 0 && e2 < s.nlat) ray_cone_roots(r, s.cth[e2], -s1, best, step);
        }
    }
    r.u_lat = best;
    r.lat_step = step;
}

__device__ __forceinline__ void ray_plane_root(const Ray& r, float cp, float sp, int step, float& best, int& best_step)
{
    const float den = fmaf(r.ny, cp, -r.nx * sp);  // n . N
    const float num = fmaf(r.pcy, cp, -r.pcx * sp);
    const float ur = -num * rcp_approx(den);        // den == 0 -> inf / nan: rejected
    if (ur > r.u && ur < best) {
        const float hx = fmaf(r.nx, ur, r.pcx), hy = fmaf(r.ny, ur, r.pcy);
        if (fmaf(hx, cp, hy * sp) > 0.0f) { best = ur; best_step = step; }  // the half-plane, not its mirror
    }
}

__device__ __forceinline__ void ray_setup_lon(Ray& r, const GeomSmem& s)
{
    float best = kInf;
    int step = 0;
    if (s.nlon > 1) {
        ray_plane_root(r, s.cph[r.k], s.sph[r.k], -1, best, step);
        ray_plane_root(r, s.cph[r.k + 1], s.sph[r.k + 1], +1, best, step);
    }
    r.u_lon = best;
    r.lon_step = step;
}

// Column pointer of (j, k) in the staged extinction table of one channel (alpha_tab points at that channel).
// DUAL: the table holds pairs (alpha, beta) per cell -- same layout, two floats per entry.
template <bool DUAL = false>
__device__ __forceinline__ const float* ray_column(const GeomSmem& s, const float* __restrict__ alpha_tab, int j, int k)
{
    return alpha_tab + ((size_t)(k * s.nlat + j) * s.col_stride + 1) * (DUAL ? 2 : 1);
}

// Extinction of the current cell and, one step ahead, of the radial neighbour the ray will enter next: the march
// loop consumes alpha one iteration after the load was issued, so the gather latency overlaps a full step.
template <bool DUAL = false>
__device__ __forceinline__ void ray_load_alpha(Ray& r, const GeomSmem& s, const float* __restrict__ alpha_tab)
{
    GCMCRT_CHECK(r.j >= 0 && r.j < s.nlat && r.k >= 0 && r.k < s.nlon && r.i >= 0 && r.i < s.nlev);
    GCMCRT_CHECK(r.rad_step == 1 || r.rad_step == -1);
    const float* colp = ray_column<DUAL>(s, alpha_tab, r.j, r.k);
    if (DUAL) {
        const float2 a = __ldg(reinterpret_cast<const float2*>(colp) + r.i);
        r.pn = colp + 2 * (r.i + r.rad_step);
        const float2 an = __ldg(reinterpret_cast<const float2*>(r.pn));
        r.alpha = a.x; r.beta = a.y; r.alpha_n = an.x; r.beta_n = an.y;
    } else {
        r.alpha = __ldg(colp + r.i);
        r.pn = colp + (r.i + r.rad_step);
        r.alpha_n = __ldg(r.pn);
    }
}

// Start a ray at p with unit direction n inside cell (i,j,k).
template <bool DUAL = false>
__device__ __forceinline__ void ray_init(Ray& r, const GeomSmem& s, float px, float py, float pz, float nx, float ny,
                                         float nz, int i, int j, int k, const float* __restrict__ alpha_tab)
{
    const float b0 = fmaf(px, nx, fmaf(py, ny, pz * nz));
    {   // d^2 = |p x n|^2 / |n|^2 in fp64, kept as a double-float: once per ray, so that every later
        // R_k^2 - d^2 is exact to fp32 rounding (fp32 products of 1e8 m coordinates carry 1e9 m^2 of error)
        const double dpx = px, dpy = py, dpz = pz, dnx = nx, dny = ny, dnz = nz;
        const double cx = dpy * dnz - dpz * dny, cy = dpz * dnx - dpx * dnz, cz = dpx * dny - dpy * dnx;
        const double eps = fma(dnx, dnx, fma(dny, dny, fma(dnz, dnz, -1.0)));   // |n|^2 - 1 ~ 1e-7
        const double cc = fma(cx, cx, fma(cy, cy, cz * cz));
        const double d2 = fma(-cc, eps * (1.0 - eps), cc);                      // cc / (1 + eps)
        r.d2 = float(d2);
        r.d2lo = float(d2 - double(r.d2));
    }
    r.pcx = fmaf(-nx, b0, px); r.pcy = fmaf(-ny, b0, py); r.pcz = fmaf(-nz, b0, pz);
    r.nx = nx; r.ny = ny; r.nz = nz;
    r.u = b0;
    r.i = i; r.j = j; r.k = k;
    ray_setup_rad(r, s);
    ray_setup_lat(r, s);
    ray_setup_lon(r, s);
    ray_load_alpha<DUAL>(r, s, alpha_tab);
}

// One step of the march, radial fast path.  tau accumulates over the segment up to the next face.  A shell crossing
// is completed here (index, next shell root, alpha rotation + prefetch) and returns RAY_FLYING; when the next face
// is a cone or a half-plane the ray is advanced to it and RAY_PARK is returned: the caller completes the crossing
// with ray_lateral().  Once a ray has crossed a shell outward it stays outward (u > 0), so only a ray still moving
// inward has to ask whether the next inner shell lies outside its impact parameter.
// DUAL (continuous absorption, Eq. 12): tau_b accumulates the second extinction over the same segments.
template <bool DUAL = false>
__device__ __forceinline__ int ray_step(Ray& r, const GeomSmem& s, float& tau, float tau_limit, float* tau_b = nullptr)
{
    const float ul = fminf(r.u_lat, r.u_lon);
    const float un = fminf(r.u_rad, ul);
    // the clamp matters: a flight that starts on a cell face in a direction nearly tangent to it (the event position is
    // rounded to fp32, 8 m at 1e8 m) can find the next roots kilometres behind its start point
    const float ds = fmaxf(un - r.u, 0.0f);
    const float tnew = fmaf(r.alpha, ds, tau);
    if (tnew >= tau_limit) {  // the limit is reached inside this cell
        const float dl = __fdividef(tau_limit - tau, r.alpha);   // MUFU.RCP + FMUL: the IEEE sequence is 20 instructions, once
        r.u += dl;                                               // per flight at a different step in every lane
        if (DUAL) *tau_b = fmaf(r.beta, dl, *tau_b);
        tau = tau_limit;
        return RAY_LIMIT;
    }
    tau = tnew;
    if (DUAL) *tau_b = fmaf(r.beta, ds, *tau_b);
    r.u = fmaxf(un, r.u);
    if (r.u_rad > ul) return RAY_PARK;  // ties: shells first (C1)
    r.i += r.rad_step;
    GCMCRT_CHECK(r.i >= -1 && r.i <= s.nlev);
    if ((unsigned)r.i >= (unsigned)s.nlev) return r.i < 0 ? RAY_SURFACE : RAY_ESCAPE;   // r.i is left outside the grid
    r.alpha = r.alpha_n;   // prefetched for exactly this cell
    if (DUAL) r.beta = r.beta_n;
    if (r.i == r.i_turn) r.rad_step = 1;   // the inner shell of this cell lies inside the impact parameter
    else r.ish += r.rad_step;              // (turning, the shell just crossed inward is the next one outward)
    // no clamp: this shell lies a whole layer beyond the one just crossed (or is the shell just crossed inward, which
    // the turn search found reachable with the same expression), so R_k^2 - d^2 > 0
    const float sq = sqrt_approx(shell_q(r, s, r.ish));
    r.u_rad = __int_as_float(__float_as_int(sq) | (r.rad_step & 0x80000000));
    r.pn += DUAL ? 2 * r.rad_step : r.rad_step;   // also right at the turn: the prefetch pointed at this cell, the next one is one up
    if (DUAL) {
        const float2 an = __ldg(reinterpret_cast<const float2*>(r.pn));
        r.alpha_n = an.x; r.beta_n = an.y;
    } else {
        r.alpha_n = __ldg(r.pn);
    }
    return RAY_FLYING;
}

// The plain-crossing loops of ray_run(), written in PTX: two crossings per trip with the roles of (alpha, alpha_n) and
// (tau, tau_new) swapping between them, so that the loop body holds no register moves (compiled from C++, ptxas spends
// 5 moves and a constant load per crossing on the loop-carried state); the exits restore the canonical state.
// DIR = +1: outward (shell address + 8, column pointer + 4 per crossing); -1: inward (the root takes the minus sign).
#define GCMCRT_RUN_LOOP(SOFF1, SOFF2, POFF1, POFF2, SSTEP1, SSTEP2, PSTEP1, PSTEP2, NEG)                              \
    asm volatile(                                                                                                      \
        "{\n\t"                                                                                                        \
        ".reg .pred p;\n\t"                                                                                            \
        ".reg .f32 ds, tn, hi, lo, q, tmp;\n\t"                                                                        \
        ".reg .s32 n1;\n\t"                                                                                            \
        "LOOP_%=:\n\t"                                                                                                 \
        "setp.ge.s32 p, %7, %12;\n\t"                                                                                  \
        "@p bra DONE_A_%=;\n\t"                                                                                        \
        "sub.f32 ds, %1, %0;\n\t"                                                                                      \
        "max.f32 ds, ds, 0f00000000;\n\t"                                                                              \
        "fma.rn.f32 tn, %2, ds, %4;\n\t"                                                                               \
        "setp.ge.f32 p, tn, %9;\n\t"                                                                                   \
        "setp.gt.or.f32 p, %1, %8, p;\n\t"                                                                             \
        "@p bra DONE_A_%=;\n\t"                                                                                        \
        "max.f32 %0, %1, %0;\n\t"                                                                                      \
        "ld.shared.v2.f32 {hi, lo}, [%6+" #SOFF1 "];\n\t"                                                              \
        "ld.global.nc.f32 %2, [%5+" #POFF1 "];\n\t"                                                                    \
        "sub.f32 hi, hi, %10;\n\t"                                                                                     \
        "sub.f32 lo, lo, %11;\n\t"                                                                                     \
        "add.f32 q, hi, lo;\n\t"                                                                                       \
        "sqrt.approx.ftz.f32 %1, q;\n\t" NEG                                                                           \
        "add.s32 n1, %7, 1;\n\t"                                                                                       \
        "setp.ge.s32 p, n1, %12;\n\t"                                                                                  \
        "@p bra DONE_B_%=;\n\t"                                                                                        \
        "sub.f32 ds, %1, %0;\n\t"                                                                                      \
        "max.f32 ds, ds, 0f00000000;\n\t"                                                                              \
        "fma.rn.f32 %4, %3, ds, tn;\n\t"                                                                               \
        "setp.ge.f32 p, %4, %9;\n\t"                                                                                   \
        "setp.gt.or.f32 p, %1, %8, p;\n\t"                                                                             \
        "@p bra DONE_B_%=;\n\t"                                                                                        \
        "max.f32 %0, %1, %0;\n\t"                                                                                      \
        "ld.shared.v2.f32 {hi, lo}, [%6+" #SOFF2 "];\n\t"                                                              \
        "ld.global.nc.f32 %3, [%5+" #POFF2 "];\n\t"                                                                    \
        "sub.f32 hi, hi, %10;\n\t"                                                                                     \
        "sub.f32 lo, lo, %11;\n\t"                                                                                     \
        "add.f32 q, hi, lo;\n\t"                                                                                       \
        "sqrt.approx.ftz.f32 %1, q;\n\t" NEG                                                                           \
        "add.s32 %6, %6, " #SSTEP2 ";\n\t"                                                                             \
        "add.s64 %5, %5, " #PSTEP2 ";\n\t"                                                                             \
        "add.s32 %7, %7, 2;\n\t"                                                                                       \
        "bra LOOP_%=;\n\t"                                                                                             \
        "DONE_B_%=:\n\t"   /* one crossing into the trip: current alpha in %3, next in %2, tau in tn */               \
        "mov.f32 tmp, %2;\n\t"                                                                                         \
        "mov.f32 %2, %3;\n\t"                                                                                          \
        "mov.f32 %3, tmp;\n\t"                                                                                         \
        "mov.f32 %4, tn;\n\t"                                                                                          \
        "add.s32 %6, %6, " #SSTEP1 ";\n\t"                                                                             \
        "add.s64 %5, %5, " #PSTEP1 ";\n\t"                                                                             \
        "add.s32 %7, %7, 1;\n\t"                                                                                       \
        "DONE_A_%=:\n\t"                                                                                               \
        "}"                                                                                                            \
        : "+f"(u), "+f"(u_rad), "+f"(alpha), "+f"(alpha_n), "+f"(tau), "+l"(pn), "+r"(sa), "+r"(n)                     \
        : "f"(ul), "f"(tau_limit), "f"(d2), "f"(d2lo), "r"(plain))

// Up to KSTEPS steps of ray_step() for a ray in flight, same arithmetic in the same order (bit-identical tau, u and
// indices), written as two runs -- inward while the ray descends, outward after it has turned (it never turns back).
// Inside a run the direction, the lateral limit min(u_lat, u_lon), the shared-memory address of the next shell and the
// column pointer are loop-carried registers, and the loop body is the plain shell crossing only: anything else (tau
// limit reached, cone / half-plane next, lower boundary, turn, top of the atmosphere) leaves the loop through ONE
// exit before any state is modified and is classified after it, once per run.  A shell crossing costs ~25 issued
// instructions instead of ~50.  nseg counts the steps taken.  Returns the ray status (RAY_FLYING: budget spent).
template <int KSTEPS>
__device__ __forceinline__ int ray_run(Ray& r, const GeomSmem& s, float& tau_io, float tau_limit, unsigned int& nseg)
{
    const float ul = fminf(r.u_lat, r.u_lon);
    const float d2 = r.d2, d2lo = r.d2lo;
    float u = r.u, u_rad = r.u_rad, alpha = r.alpha, alpha_n = r.alpha_n, tau = tau_io;
    const float* pn = r.pn;
    uint32_t sa = s.r2_saddr + 8u * uint32_t(r.ish);     // shared-space address of R2[ish]
    const uint32_t sa0 = s.r2_saddr;
    int status = RAY_FLYING, n = 0;
    bool inward = r.rad_step < 0;
    asm volatile("" : "+f"(tau_limit));   // a register, not a constant-bank load per step
    if (inward) {
        // crossing shell sa_stop inward is no plain crossing: it enters the turning cell i_turn (the shell just crossed
        // is then the next one outward) or, for a ray that does not turn inside the grid, leaves through the lower boundary
        const uint32_t sa_stop = s.r2_saddr + 8u * uint32_t(max(r.i_turn + 1, 0));
        const int plain = min(KSTEPS, int((sa - sa_stop) >> 3));   // plain crossings before that one, within the budget
        GCMCRT_RUN_LOOP(-8, -16, -4, -8, -8, -16, -4, -8, "neg.f32 %1, %1;\n\t");   // plain inward crossings
        if (n < KSTEPS) {
            ++n;
            const float un = fminf(u_rad, ul);
            const float tnew = fmaf(alpha, fmaxf(un - u, 0.0f), tau);
            if (tnew >= tau_limit) {
                u += __fdividef(tau_limit - tau, alpha);
                tau = tau_limit; status = RAY_LIMIT;
            } else {
                tau = tnew;
                u = fmaxf(un, u);
                if (u_rad > ul) status = RAY_PARK;                        // ties: shells first (C1)
                else if (r.i_turn < 0) status = RAY_SURFACE;              // sa == sa0: the cell index leaves the grid
                else {                                                    // the turn
                    alpha = alpha_n;
                    inward = false;
                    float hi, lo;
                    asm("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(hi), "=f"(lo) : "r"(sa));
                    u_rad = sqrt_approx((hi - d2) + (lo - d2lo));
                    ++pn;
                    alpha_n = __ldg(pn);
                }
            }
        }
    }
    if (!inward && status == RAY_FLYING) {
        const uint32_t sa_top = s.r2_saddr + 8u * uint32_t(s.nlev);
        const int plain = min(KSTEPS, n + int((sa_top - sa) >> 3));   // plain crossings before the one that leaves the grid
        GCMCRT_RUN_LOOP(8, 16, 4, 8, 8, 16, 4, 8, "");   // plain outward crossings
        if (n < KSTEPS) {
            ++n;
            const float un = fminf(u_rad, ul);
            const float tnew = fmaf(alpha, fmaxf(un - u, 0.0f), tau);
            if (tnew >= tau_limit) {
                u += __fdividef(tau_limit - tau, alpha);
                tau = tau_limit; status = RAY_LIMIT;
            } else {
                tau = tnew;
                u = fmaxf(un, u);
                status = u_rad > ul ? RAY_PARK : RAY_ESCAPE;              // sa == sa_top: i = nlev
            }
        }
    }
    const int ish = int((sa - sa0) >> 3);
    GCMCRT_CHECK(sa >= sa0 && ish >= 0 && ish <= s.nlev && n >= 0 && n <= KSTEPS);
    GCMCRT_CHECK(status == RAY_SURFACE || status == RAY_ESCAPE || (ish - (inward ? 0 : 1) >= 0 && ish - (inward ? 0 : 1) < s.nlev));
    r.ish = ish;
    r.i = status == RAY_SURFACE ? -1 : (status == RAY_ESCAPE || inward ? ish : ish - 1);
    r.rad_step = inward ? -1 : 1;
    r.u = u; r.u_rad = u_rad; r.alpha = alpha; r.alpha_n = alpha_n; r.pn = pn;
    tau_io = tau;
    nseg += n;
    return status;
}

// Completes the cone / half-plane crossing of a parked ray (ties: cones before planes, C1).
template <bool DUAL = false>
__device__ __forceinline__ void ray_lateral(Ray& r, const GeomSmem& s, const float* __restrict__ alpha_tab)
{
    if (r.u_lat <= r.u_lon) {
        r.j = min(max(r.j + r.lat_step, 0), s.nlat - 1);
        ray_setup_lat(r, s);
    } else {
        r.k += r.lon_step;
        r.k = (r.k < 0) ? r.k + s.nlon : (r.k >= s.nlon ? r.k - s.nlon : r.k);
        // the azimuth of a straight line is monotonic: the next half-plane lies in the same direction
        float best = kInf;
        int step = 0;
        const int e = r.lon_step > 0 ? r.k + 1 : r.k;
        ray_plane_root(r, s.cph[e], s.sph[e], r.lon_step, best, step);
        r.u_lon = best;
        r.lon_step = step == 0 ? r.lon_step : step;
    }
    ray_load_alpha<DUAL>(r, s, alpha_tab);
}

__device__ __forceinline__ void ray_position(const Ray& r, float& px, float& py, float& pz)
{
    px = fmaf(r.nx, r.u, r.pcx); py = fmaf(r.ny, r.u, r.pcy); pz = fmaf(r.nz, r.u, r.pcz);
}

// Binary search: cell m with e[m] <= x < e[m+1] (ascending edges), clamped.
__device__ __forceinline__ int locate_ascending(const float* e, int n, float x)
{
    int lo = 0, hi = n;  // invariant: e[lo] <= x < e[hi] after clamping
    while (hi - lo > 1) {
        const int mid = (lo + hi) >> 1;
        if (x >= e[mid]) lo = mid; else hi = mid;
    }
    return lo;
}
// Same for descending tables (cosines of ascending colatitudes).
__device__ __forceinline__ int locate_descending(const float* e, int n, float x)
{
    int lo = 0, hi = n;
    while (hi - lo > 1) {
        const int mid = (lo + hi) >> 1;
        if (x <= e[mid]) lo = mid; else hi = mid;
    }
    return lo;
}

__device__ __forceinline__ void locate_angles(const GeomSmem& s, float px, float py, float pz, int& j, int& k)
{
    j = 0; k = 0;
    if (s.nlat > 1) {
        const float ct = pz * rsqrtf(fmaf(px, px, fmaf(py, py, pz * pz)));
        j = locate_descending(s.cth, s.nlat, ct);
    }
    if (s.nlon > 1) {
        float phi = atan2f(py, px);
        if (phi < 0.0f) phi += 2.0f * kPi;
        k = locate_ascending(s.ph, s.nlon, phi);
    }
}

}  // namespace gcmcrt

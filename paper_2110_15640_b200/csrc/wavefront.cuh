// wavefront.cuh -- generation-synchronous transport (A3-A6, A8): the bulk of every pass runs as a short sequence of
// kernels in which all lanes of a warp do the same thing at the same time, instead of one persistent kernel whose
// lanes are each somewhere else in a packet's life.
//
//   wave_launch_keys_kernel   albedo: entry column of every fresh packet (Philox block 0)          -> sort (sort.cuh)
//   wave_first_flight_kernel  albedo: launch (O3) + first flight, packets in entry-column order: 32 parallel rays
//                             per warp that enter the same column at the top of the atmosphere
//   wave_emit_kernel          emission: emitting cell ~ L_i (Eq. 13), point in the cell (O4)      -> generation 0
//   wave_interact_kernel      generation g -> g+1: for every event record of generation g: absorb / scatter (O6, O7,
//                             Eq. 6, Eq. 8), then the survivors -- compacted through a warp-private shared-memory
//                             stage so that the expensive half runs on full warps -- fly to their next event
//
// The event buffer is the queue: a record holds the packet's whole state at the event (kernels.cuh EventBuf), each
// generation appends the next one behind itself, and the peel kernel later integrates all of them.  After a fixed
// number of generations the few packets still alive are parked in the suspended list and finished by the persistent
// transport_kernel (kernels.cuh), which is also what resumes packets that did not fit into a full event buffer.
// The arithmetic per packet is identical to the persistent kernel's (same Philox blocks, same ray code), so
// per-packet event counts do not depend on which of the two carried a packet.
#pragma once

namespace gcmcrt {

constexpr int kWaveThreads = 256;
constexpr int kStageFields = 14;
constexpr int kStageSlots = 64;   // per warp: at most 31 left over + 32 new survivors
constexpr int kLaunchTauBuckets = 16;   // launch order: packets of one entry column grouped by sampled optical depth

struct WaveConst {
    const unsigned int* perm;      // albedo: launch order, perm[t] in [0, n_items)
    unsigned int* keys;            // albedo: launch sort keys [n_items]
    unsigned int* lhist;           // albedo: histogram of the launch sort keys, counted by the key kernel
    const unsigned int* gen_mark;  // interact: events [gen_mark[0], gen_mark[1]) form this generation (device)
    int park_all;                  // last generation: survivors' next events go to the suspended list
    int c_fold;                    // launch sort key window (its first channel is PassCtrl::chan_lo)
    float* flights;                // interact: per-warp lists of flights in progress [n_warps][kFlightFields][kStageSlots]
};

struct WaveCounters {
    unsigned long long events = 0, seg = 0, esc = 0, abs = 0, surf = 0, stuck = 0;
    double escw = 0.0;
};

__device__ __forceinline__ void wave_flush_counters(const RunConst& rc, WaveCounters& c)
{
    c.events = warp_sum_u64(c.events); c.seg = warp_sum_u64(c.seg); c.esc = warp_sum_u64(c.esc);
    c.abs = warp_sum_u64(c.abs); c.surf = warp_sum_u64(c.surf); c.stuck = warp_sum_u64(c.stuck);
    c.escw = warp_sum_f64(c.escw);
    if (lane_id() == 0) {
        if (c.events) atomicAdd(&rc.counters->events, c.events);
        if (c.seg) atomicAdd(&rc.counters->seg_transport, c.seg);
        if (c.esc) atomicAdd(&rc.counters->escaped, c.esc);
        if (c.abs) atomicAdd(&rc.counters->absorbed, c.abs);
        if (c.surf) atomicAdd(&rc.counters->surface, c.surf);
        if (c.stuck) atomicAdd(&rc.counters->stuck, c.stuck);
        if (c.escw != 0.0) atomicAdd(&rc.counters->escaped_weight, c.escw);
    }
}

// peel-off points a packet has made before an event of `kind` that follows m_inter completed interactions
__device__ __forceinline__ uint32_t nev_before(const RunConst& rc, uint32_t kind, uint32_t m_inter)
{
    return m_inter + ((rc.mode == 1 && kind != EV_EMIT) ? 1u : 0u);
}

__device__ __forceinline__ void wave_finish_packet(const RunConst& rc, uint32_t chan_run, uint32_t pkt, uint32_t nev)
{
    GCMCRT_CHECK(chan_run < (uint32_t)rc.n_chan_run && pkt >= rc.pkt_begin && pkt - rc.pkt_begin < rc.n_pkt);
    if (rc.event_count) rc.event_count[(size_t)chan_run * rc.n_pkt + (pkt - rc.pkt_begin)] = nev;
}

// Warp-collective.  Lanes with `want` append an event record (one atomic per warp); when the buffer is full, or in
// the last generation, the packet is parked at the event instead (not yet recorded), in the persistent kernel's format.
// (rx, ry, rz) is what the record stores as direction (incoming direction, or the surface normal), (dx, dy, dz) the
// packet's flight direction.
__device__ __forceinline__ bool wave_record(const RunConst& rc, const EventBuf& ev, const SuspBuf& susp, int park_all,
                                            bool want, uint32_t kind, float px, float py, float pz, float rx, float ry,
                                            float rz, float dx, float dy, float dz, float W, uint32_t cellp,
                                            uint32_t chan_run, uint32_t pkt, uint32_t m_inter, WaveCounters& wcnt)
{
    const unsigned m = __ballot_sync(kFullMask, want);
    if (m == 0) return false;
    unsigned int slot = 0xffffffffu;
    if (!park_all) {
        unsigned int base = 0;
        if (lane_id() == __ffs(m) - 1) base = atomicAdd(ev.count, (unsigned)__popc(m));
        base = __shfl_sync(kFullMask, base, __ffs(m) - 1);
        slot = base + rank_in_mask(m);
    }
    if (want) {
        if (slot < ev.cap) {
            const uint32_t meta = kind | batch_of(rc, pkt) << 2 | chan_run << 8;
            float4 prop = make_float4(0.f, 0.f, 0.f, 0.f);
            if (kind == EV_MEDIUM) {   // the cell's scattering properties travel with the record
                const int i = cellp & 1023, j = (cellp >> 10) & 1023, k = cellp >> 20;
                prop = __ldg(rc.prop + (size_t)(rc.chan_begin + int(chan_run)) * rc.geom.ncell +
                             ((k * rc.geom.nlat + j) * rc.geom.nlev + i));
            }
            write_event(ev, slot, px, py, pz, W, rx, ry, rz, m_inter, cellp, meta, pkt, prop);
            ++wcnt.events;
        } else {
            const unsigned int sidx = atomicAdd(susp.count, 1u);
            if (sidx < susp.cap) {
                susp.s0[sidx] = make_float4(px, py, pz, W);
                susp.s1[sidx] = make_float4(dx, dy, dz, __uint_as_float(cellp));
                susp.s2[sidx] = make_uint4(chan_run, pkt, m_inter, nev_before(rc, kind, m_inter) | kind << 28);
            } else {
                ++wcnt.stuck;
            }
        }
    }
    return want && slot < ev.cap;   // true: the event is in the buffer (false: parked, the persistent kernel records it)
}

// Warp-collective: marches every lane whose status is RAY_FLYING / RAY_PARK for at most `budget` steps (radial steps,
// cone / half-plane crossings batched across the warp).  Returns the number of loop steps spent (warp-uniform).
template <int KSTEPS>
__device__ __forceinline__ int wave_march(const RunConst& rc, const GeomSmem& gs, int& st, Ray& ray, float& tau,
                                          float tau_t, const float* alpha_c, int budget, WaveCounters& wcnt)
{
    unsigned int seg32 = 0;
    int it = 0;
    for (; it < budget; it += KSTEPS) {
        const unsigned m_fly = __ballot_sync(kFullMask, st == RAY_FLYING);
        const unsigned m_park = __ballot_sync(kFullMask, st == RAY_PARK);
        if ((m_fly | m_park) == 0) break;
        if (m_park && (__popc(m_park) >= rc.t_lateral || m_fly == 0)) {
            if (st == RAY_PARK) {
                ray_lateral(ray, gs, alpha_c);
                st = RAY_FLYING;
            }
        }
        if (st == RAY_FLYING) st = ray_run<KSTEPS>(ray, gs, tau, tau_t, seg32);   // lanes in flight step together
    }
    wcnt.seg += seg32;
    return it;
}

// Warp-collective: lanes with `fin` have ended their flight with status st: record the next event (or park the
// packet), or close the packet.
__device__ __forceinline__ void wave_close(const RunConst& rc, const EventBuf& ev, const SuspBuf& susp, int park_all,
                                           bool fin, int st, const Ray& ray, float W, float tau, uint32_t chan_run,
                                           uint32_t pkt, uint32_t m_inter, WaveCounters& wcnt)
{
    if (fin) W *= stretch_weight(rc, st, tau);   // path length stretching: the weight of the flight's outcome
    const bool surf_ev = fin && st == RAY_SURFACE && rc.surface_albedo > 0.f;
    const bool want = fin && (st == RAY_LIMIT || surf_ev);
    float px = 0.f, py = 0.f, pz = 0.f, rx = ray.nx, ry = ray.ny, rz = ray.nz;
    if (want) {
        ray_position(ray, px, py, pz);
        if (surf_ev) {
            const float rn = rsqrtf(fmaf(px, px, fmaf(py, py, pz * pz)));
            rx = px * rn; ry = py * rn; rz = pz * rn;
        }
    }
    wave_record(rc, ev, susp, park_all, want, surf_ev ? EV_SURFACE : EV_MEDIUM, px, py, pz, rx, ry, rz, ray.nx, ray.ny,
                ray.nz, W, pack_cell(surf_ev ? 0 : ray.i, ray.j, ray.k), chan_run, pkt, m_inter, wcnt);
    if (fin && !want) {
        if (st == RAY_ESCAPE) { ++wcnt.esc; wcnt.escw += double(W); }
        else if (st == RAY_SURFACE) ++wcnt.surf;
        else ++wcnt.stuck;
        wave_finish_packet(rc, chan_run, pkt, m_inter + (rc.mode == 1 ? 1u : 0u));
    }
}

// Warp-collective: 32 flights that start together, each marched to its end.
template <int KSTEPS>
__device__ __forceinline__ void wave_fly(const RunConst& rc, const EventBuf& ev, const SuspBuf& susp, int park_all,
                                         const GeomSmem& gs, bool active, Ray& ray, float tau_t, const float* alpha_c,
                                         float W, uint32_t chan_run, uint32_t pkt, uint32_t m_inter, WaveCounters& wcnt)
{
    int st = active ? RAY_FLYING : RAY_NONE;
    float tau = 0.f;
    wave_march<KSTEPS>(rc, gs, st, ray, tau, tau_t, alpha_c, rc.geom.maxseg + 1, wcnt);
    if (active && (st == RAY_FLYING || st == RAY_PARK)) st = RAY_STUCK;   // step budget exhausted
    wave_close(rc, ev, susp, park_all, active, st, ray, W, tau, chan_run, pkt, m_inter, wcnt);
}

// ---- flights in progress, set aside (interact kernel): a scattered packet's flight is short most of the time and
// long now and then, so a warp marches its 32 fresh flights for a few steps only and moves the unfinished ones to a
// per-warp list in global memory (L2-resident); 32 of those are then marched together for longer.  23 words per flight.
constexpr int kFlightFields = 23;
constexpr int kInteractK = 8;   // steps per ray_run call in the interact kernel
constexpr int kFirstRoundSteps = 8, kLongRoundSteps = 16;   // measured: (4, 16) 57.9 ms, (8, 16) 56.6, (16, 32) 58.1, (2, 8) 60.8

__device__ __forceinline__ void flight_save(float* fl, const Ray& r, float tau, float tau_t, float W, uint32_t chan_run,
                                            uint32_t pkt, uint32_t m_inter, int st, int used)
{
    fl[0 * kStageSlots] = r.pcx; fl[1 * kStageSlots] = r.pcy; fl[2 * kStageSlots] = r.pcz;
    fl[3 * kStageSlots] = r.nx; fl[4 * kStageSlots] = r.ny; fl[5 * kStageSlots] = r.nz;
    fl[6 * kStageSlots] = r.d2; fl[7 * kStageSlots] = r.d2lo; fl[8 * kStageSlots] = r.u;
    fl[9 * kStageSlots] = r.u_rad; fl[10 * kStageSlots] = r.u_lat; fl[11 * kStageSlots] = r.u_lon;
    fl[12 * kStageSlots] = r.alpha; fl[13 * kStageSlots] = r.alpha_n;
    fl[14 * kStageSlots] = tau; fl[15 * kStageSlots] = tau_t; fl[16 * kStageSlots] = W;
    fl[17 * kStageSlots] = __uint_as_float(pack_cell(r.i, r.j, r.k));
    const uint32_t steps = uint32_t(r.rad_step + 1) | uint32_t(r.lat_step + 1) << 2 | uint32_t(r.lon_step + 1) << 4 |
                           uint32_t(st == RAY_PARK) << 6 | uint32_t(used) << 8;
    fl[18 * kStageSlots] = __uint_as_float(steps);
    fl[19 * kStageSlots] = __uint_as_float(chan_run); fl[20 * kStageSlots] = __uint_as_float(pkt);
    fl[21 * kStageSlots] = __uint_as_float(m_inter);
    fl[22 * kStageSlots] = __int_as_float(r.i_turn);
}

__device__ __forceinline__ void flight_load(const float* fl, const RunConst& rc, const GeomSmem& gs, Ray& r, float& tau,
                                            float& tau_t, float& W, uint32_t& chan_run, uint32_t& pkt, uint32_t& m_inter,
                                            int& st, int& used, const float*& alpha_c)
{
    r.pcx = fl[0 * kStageSlots]; r.pcy = fl[1 * kStageSlots]; r.pcz = fl[2 * kStageSlots];
    r.nx = fl[3 * kStageSlots]; r.ny = fl[4 * kStageSlots]; r.nz = fl[5 * kStageSlots];
    r.d2 = fl[6 * kStageSlots]; r.d2lo = fl[7 * kStageSlots]; r.u = fl[8 * kStageSlots];
    r.u_rad = fl[9 * kStageSlots]; r.u_lat = fl[10 * kStageSlots]; r.u_lon = fl[11 * kStageSlots];
    r.alpha = fl[12 * kStageSlots]; r.alpha_n = fl[13 * kStageSlots];
    tau = fl[14 * kStageSlots]; tau_t = fl[15 * kStageSlots]; W = fl[16 * kStageSlots];
    unpack_cell(__float_as_uint(fl[17 * kStageSlots]), r.i, r.j, r.k);
    const uint32_t steps = __float_as_uint(fl[18 * kStageSlots]);
    r.rad_step = int(steps & 3u) - 1; r.lat_step = int((steps >> 2) & 3u) - 1; r.lon_step = int((steps >> 4) & 3u) - 1;
    st = (steps >> 6) & 1u ? RAY_PARK : RAY_FLYING;
    used = int(steps >> 8);
    chan_run = __float_as_uint(fl[19 * kStageSlots]); pkt = __float_as_uint(fl[20 * kStageSlots]);
    m_inter = __float_as_uint(fl[21 * kStageSlots]);
    r.i_turn = __float_as_int(fl[22 * kStageSlots]);
    r.ish = r.rad_step > 0 ? r.i + 1 : r.i;
    alpha_c = rc.alpha + (size_t)(rc.chan_begin + int(chan_run)) * rc.geom.alpha_stride;
    r.pn = ray_column(gs, alpha_c, r.j, r.k) + (r.i + r.rad_step);
}

// O3: uniform point on the star-facing TOA disc from Philox block (event 0, purpose 0), and its entry column
// (Sect. 5.1 with multiple scattering: the start of the packet's transit chord instead; returns false for a chord off
// the stellar disc, which carries no light)
template <bool LOCATE = true>
__device__ __forceinline__ bool albedo_launch_point(const RunConst& rc, const GeomSmem& gs, const Zeta4& z, float& px,
                                                    float& py, float& pz, int& j, int& k)
{
    bool lit = true;
    if (rc.launch_chord) {
        float b, X, Y, Wld;
        chord_point(rc, z.z0, z.z1, b, X, Y, Wld);
        chord_start(rc, b, X, Y, px, py, pz);
        lit = Wld > 0.f;
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
    if (LOCATE) locate_angles(gs, px, py, pz, j, k);
    return lit;
}

__device__ __forceinline__ void wave_item(const RunConst& rc, unsigned long long item, uint32_t& chan_run, uint32_t& pkt)
{
    chan_run = uint32_t(div_magic(item, rc.n_pkt, rc.magic_npkt));
    pkt = rc.pkt_begin + uint32_t(item - (unsigned long long)chan_run * rc.n_pkt);
}

// albedo: sort key of every fresh packet = (channel window slot, entry column, optical-depth bucket)
__global__ void __launch_bounds__(kWaveThreads) wave_launch_keys_kernel(const __grid_constant__ RunConst rc,
                                                                       const WaveConst wc)
{
    extern __shared__ float smem_f[];
    const GeomSmem gs = load_geom(rc.geom, smem_f);
    __syncthreads();
    const unsigned int n_items = rc.ctrl->n_fresh;
    const unsigned long long item0 = rc.ctrl->item0;
    const int chan_lo = rc.ctrl->chan_lo;
    for (unsigned int t = blockIdx.x * blockDim.x + threadIdx.x; t < n_items; t += gridDim.x * blockDim.x) {
        uint32_t chan_run, pkt;
        wave_item(rc, item0 + t, chan_run, pkt);
        const uint32_t ckey = rc.chan_key0 + uint32_t(rc.chan_begin) + chan_run;
        const Zeta4 z = zeta_block(rc.seed, ckey, pkt, 0, 0);
        float px, py, pz;
        int j, k;
        albedo_launch_point(rc, gs, z, px, py, pz, j, k);
        const int slot = min(max(int(chan_run) - chan_lo, 0), wc.c_fold - 1);
        // the extinction grows roughly exponentially with depth, so the level a packet reaches goes with log(tau):
        // packets of one column that share a log2(tau) bucket end their first flight within a few cells of each other
        const float lt = __log2f(-__logf(z.z2));                       // log2 of the sampled optical depth, about -23 .. 4
        const int tb = min(max(int(floorf((lt + 8.0f) * (kLaunchTauBuckets / 12.0f))), 0), kLaunchTauBuckets - 1);
        const unsigned int key = (unsigned int)((slot * (gs.nlat * gs.nlon) + k * gs.nlat + j) * kLaunchTauBuckets + tb);
        wc.keys[t] = key;
        atomicAdd(wc.lhist + key, 1u);
    }
}

// albedo: launch + first flight, 32 packets of neighbouring entry columns per warp
template <int KSTEPS, bool FORCED>
__global__ void __launch_bounds__(kWaveThreads, FORCED ? 3 : 4)
wave_first_flight_kernel(const __grid_constant__ RunConst rc, const EventBuf ev, const SuspPair susp2, const WaveConst wc)
{
    extern __shared__ float smem_f[];
    const GeomSmem gs = load_geom(rc.geom, smem_f);
    __syncthreads();
    const SuspBuf susp = susp_select(susp2, rc.ctrl->cur);
    const unsigned int n_items = rc.ctrl->n_fresh;
    const unsigned long long item0 = rc.ctrl->item0;
    WaveCounters wcnt;
    const unsigned int warp0 = (blockIdx.x * blockDim.x + threadIdx.x) & ~31u;
    for (unsigned int base = warp0; base < n_items; base += gridDim.x * blockDim.x) {
        const unsigned int t = base + lane_id();
        const bool active = t < n_items;
        uint32_t chan_run = 0, pkt = 0;
        Ray ray{};
        float tau_t = 0.f, z2 = 0.f;
        bool lit = true;
        const float* alpha_c = rc.alpha;
        if (active) {
            const unsigned int it = __ldg(wc.perm + t);
            wave_item(rc, item0 + it, chan_run, pkt);
            const int ctab = rc.chan_begin + int(chan_run);
            alpha_c = rc.alpha + (size_t)ctab * rc.geom.alpha_stride;
            const Zeta4 z = zeta_block(rc.seed, rc.chan_key0 + uint32_t(ctab), pkt, 0, 0);
            float px, py, pz;
            // the entry column was located when the launch key was made: read it back instead of locating again
            const unsigned int col = (__ldg(wc.keys + it) / kLaunchTauBuckets) % (unsigned int)(gs.nlat * gs.nlon);
            int j = int(col % (unsigned int)gs.nlat), k = int(col / (unsigned int)gs.nlat);
            lit = albedo_launch_point<false>(rc, gs, z, px, py, pz, j, k);
            tau_t = -logf(z.z2);
            z2 = z.z2;
            ray_init(ray, gs, px, py, pz, rc.launch_dir[0], rc.launch_dir[1], rc.launch_dir[2], gs.nlev - 1, j, k, alpha_c);
        }
        float W = 1.0f;
        bool fly = active;
        if (active && !lit) {   // a transit chord off the stellar disc: the packet ends with no event
            wave_finish_packet(rc, chan_run, pkt, 0u);
            fly = false;
        }
        const bool probe_on = fly;
        bool forced = false;
        if (FORCED) {
            // Sect. 4.2 (L179), forced first scattering: the extra ray trace to the end of the grid gives tau_edge; the
            // flight is drawn from the exponential law truncated there and the packet carries 1 - e^-tau_edge.  A ray
            // that ends on a reflecting lower boundary stays analog.
            Ray probe = ray;
            int st = probe_on ? RAY_FLYING : RAY_NONE;
            float tau_e = 0.f;
            WaveCounters unused;
            wave_march<KSTEPS>(rc, gs, st, probe, tau_e, kInf, alpha_c, rc.geom.maxseg + 1, unused);
            if (probe_on && (st == RAY_ESCAPE || (st == RAY_SURFACE && !(rc.surface_albedo > 0.f)))) {
                const float pint = -expm1f(-rc.stretch * tau_e);   // stretch < 1: the hybrid with path length stretching
                if (!(pint > 0.f)) {   // empty path: the packet ends with no event
                    if (st == RAY_ESCAPE) { ++wcnt.esc; wcnt.escw += 1.0; } else ++wcnt.surf;
                    wave_finish_packet(rc, chan_run, pkt, 0u);
                    fly = false;
                } else {
                    if (st == RAY_ESCAPE) wcnt.escw += double(expf(-tau_e));   // the part that leaves without interacting
                    W = pint;
                    tau_t = -log1pf(-z2 * pint) * rc.inv_stretch;
                    forced = true;
                }
            }
        }
        if (!forced) tau_t *= rc.inv_stretch;   // path length stretching: tau = -ln(zeta) / a
        wave_fly<KSTEPS>(rc, ev, susp, wc.park_all, gs, fly, ray, tau_t, alpha_c, W, chan_run, pkt, 0u, wcnt);
    }
    wave_flush_counters(rc, wcnt);
}

// emission: generation 0 = the emission points (O4).  Eq. 13 with the composite bias xi (C10).
__global__ void __launch_bounds__(kWaveThreads, 5) wave_emit_kernel(const __grid_constant__ RunConst rc, const EventBuf ev,
                                                                const SuspPair susp2, const WaveConst wc)
{
    extern __shared__ float smem_f[];
    const GeomSmem gs = load_geom(rc.geom, smem_f);
    __syncthreads();
    const SuspBuf susp = susp_select(susp2, rc.ctrl->cur);
    const unsigned int n_items = rc.ctrl->n_fresh;
    const unsigned long long item0 = rc.ctrl->item0;
    WaveCounters wcnt;
    const unsigned int warp0 = (blockIdx.x * blockDim.x + threadIdx.x) & ~31u;
    for (unsigned int base = warp0; base < n_items; base += gridDim.x * blockDim.x) {
        const unsigned int t = base + lane_id();
        bool live = false;
        uint32_t chan_run = 0, pkt = 0, cellp = 0;
        float px = 0.f, py = 0.f, pz = 0.f, W = 1.0f;
        if (t < n_items) {
            wave_item(rc, item0 + t, chan_run, pkt);
            const int ctab = rc.chan_begin + int(chan_run);
            const Zeta4 z = zeta_block(rc.seed, rc.chan_key0 + uint32_t(ctab), pkt, 0, 0);
            const int ncell = rc.geom.ncell;
            const double* cum = rc.Lcum + (size_t)ctab * ncell;
            const double Ltot = rc.Ltot[ctab];
            int cell = 0;
            live = Ltot > 0.0;
            if (live) {
                if (double(z.z0) < rc.xi) {
                    cell = min(int(floor(double(z.z0) / rc.xi * ncell)), ncell - 1);
                } else {
                    const double frac = (double(z.z0) - rc.xi) / (1.0 - rc.xi);
                    const double x = frac * Ltot;
                    const int gi = min(int(frac * double(kEmisGuide)), kEmisGuide - 1);
                    const int* gd = rc.guide + (size_t)ctab * kEmisGuide;
                    const int lo = __ldg(gd + gi), hi = gi + 1 < kEmisGuide ? __ldg(gd + gi + 1) : ncell - 1;
                    cell = emis_search(cum, rc.Lcol + (size_t)ctab * (gs.nlat * gs.nlon), Ltot, gs.nlev, gs.nlat * gs.nlon, lo, hi, x);
                }
                if (rc.xi > 0.0) {
                    const double Li = rc.Lcell[(size_t)ctab * ncell + cell];
                    live = Li > 0.0;
                    W = live ? float(1.0 / ((1.0 - rc.xi) + rc.xi * Ltot / (double(ncell) * Li))) : 0.f;
                }
            }
            if (live) {
                GCMCRT_CHECK(cell >= 0 && cell < rc.geom.ncell);
                const int i = cell % gs.nlev, j = (cell / gs.nlev) % gs.nlat, k = cell / (gs.nlev * gs.nlat);
                const float r = gs.R[i] * cbrtf(fmaf(z.z1, gs.qcube[i], 1.0f));
                const float ct = fmaf(z.z2, gs.cth[j + 1] - gs.cth[j], gs.cth[j]);
                const float sth = sqrtf(fmaxf(0.f, 1.0f - ct * ct));
                const float phi = fmaf(z.z3, gs.ph[k + 1] - gs.ph[k], gs.ph[k]);
                float sp, cp;
                sincosf(phi, &sp, &cp);
                px = r * sth * cp; py = r * sth * sp; pz = r * ct;
                cellp = pack_cell(i, j, k);
            } else {
                wave_finish_packet(rc, chan_run, pkt, 0u);   // a packet without luminosity makes no event
            }
        }
        const bool recorded = wave_record(rc, ev, susp, wc.park_all, live, EV_EMIT, px, py, pz, 0.f, 0.f, 1.f, 0.f, 0.f, 1.f,
                                          W, cellp, chan_run, pkt, 0u, wcnt);
        if (recorded && !rc.scatter_on) {   // L210: only the initial peel-off; no generation kernel has to look at it
            ++wcnt.abs;
            wave_finish_packet(rc, chan_run, pkt, 1u);
        }
    }
    wave_flush_counters(rc, wcnt);
}

// generation g -> g + 1
// FORCED: forced scattering at every flight (forced_scatter = 2): an instance of its own, so that the default one
// carries no call to the edge probe
template <int KSTEPS, bool FORCED>
__global__ void __launch_bounds__(kWaveThreads, 3)
wave_interact_kernel(const __grid_constant__ RunConst rc, const EventBuf ev, const SuspPair susp2, const WaveConst wc)
{
    extern __shared__ float smem_f[];
    const GeomSmem gs = load_geom(rc.geom, smem_f);
    const SuspBuf susp = susp_select(susp2, rc.ctrl->cur);
    // survivors of the absorb / scatter decision wait here until a full warp of them has gathered
    float* stage = smem_f + ((rc.geom.tab_floats + 31) & ~31) + (threadIdx.x >> 5) * (kStageFields * kStageSlots);
    __syncthreads();
    WaveCounters wcnt;
    const unsigned int begin = wc.gen_mark[0], end = min(wc.gen_mark[1], ev.cap);
    const unsigned int warp0 = begin + ((blockIdx.x * blockDim.x + threadIdx.x) & ~31u);
    int staged = 0, in_flight = 0;   // warp-uniform list lengths
    float* flights = wc.flights + (size_t)((blockIdx.x * blockDim.x + threadIdx.x) >> 5) * (kFlightFields * kStageSlots);

    for (unsigned int base = warp0;; base += gridDim.x * blockDim.x) {
        const bool more = base < end;   // warp-uniform
        if (more) {
            // ---------------- phase 1: absorb or scatter (O6 / O7 / emission launch direction) ----------------
            const unsigned int e = base + lane_id();
            bool surv = false;
            float4 a = make_float4(0.f, 0.f, 0.f, 0.f), b = a;
            float ct = 0.f, zpsi = 0.f, tau_t = 0.f;
            uint32_t m_new = 0, cellp = 0, meta = 0, pkt = 0;
            if (e < end) {
                const float4* r = ev.rec + 4 * (size_t)e;
                a = r[0]; b = r[1];
                const float4 c = r[2], pr = r[3];
                const uint32_t m_inter = __float_as_uint(c.x);
                cellp = __float_as_uint(c.y); meta = __float_as_uint(c.z); pkt = __float_as_uint(c.w);
                const uint32_t kind = meta & 3u, chan_run = meta >> 8;
                const int ctab = rc.chan_begin + int(chan_run);
                const uint32_t ckey = rc.chan_key0 + uint32_t(ctab);
                const uint32_t nev = nev_before(rc, kind, m_inter) + 1u;   // peel-off points including this one
                m_new = m_inter;
                if (kind == EV_MEDIUM) {
                    m_new = m_inter + 1;
                    const Zeta4 z = zeta_block(rc.seed, ckey, pkt, m_new, 1);
                    if ((rc.max_events && int(m_new) == rc.max_events) || !rc.scatter_on ||
                        !medium_interaction(rc, pr, z, ckey, pkt, m_new, a.w, ct)) {
                        ++wcnt.abs; wave_finish_packet(rc, chan_run, pkt, nev);       // L192: absorbed
                    } else {
                        zpsi = z.z2; tau_t = -logf(z.z3); surv = true;
                    }
                } else if (kind == EV_EMIT) {
                    if (!rc.scatter_on) {
                        ++wcnt.abs; wave_finish_packet(rc, chan_run, pkt, nev);
                    } else {
                        const Zeta4 z = zeta_block(rc.seed, ckey, pkt, 1, 0);
                        ct = fmaf(2.0f, z.z0, -1.0f);   // Eq. 2
                        zpsi = z.z1; tau_t = -logf(z.z2); surv = true;
                    }
                } else {  // Lambert surface (O7, Eq. 3-4); b holds the surface normal
                    m_new = m_inter + 1;
                    const Zeta4 z = zeta_block(rc.seed, ckey, pkt, m_new, 3);
                    if (rc.max_events && int(m_new) == rc.max_events) {
                        ++wcnt.abs; wave_finish_packet(rc, chan_run, pkt, nev);
                    } else if (z.z0 >= rc.surface_albedo) {
                        ++wcnt.surf; wave_finish_packet(rc, chan_run, pkt, nev);
                    } else {
                        ct = sqrtf(z.z1); zpsi = z.z2; tau_t = -logf(z.z3); surv = true;
                    }
                }
            }
            const unsigned m_s = __ballot_sync(kFullMask, surv);
            if (surv) {
                float* sl = stage + staged + rank_in_mask(m_s);
                sl[0 * kStageSlots] = a.x; sl[1 * kStageSlots] = a.y; sl[2 * kStageSlots] = a.z; sl[3 * kStageSlots] = a.w;
                sl[4 * kStageSlots] = b.x; sl[5 * kStageSlots] = b.y; sl[6 * kStageSlots] = b.z;
                sl[7 * kStageSlots] = ct; sl[8 * kStageSlots] = zpsi; sl[9 * kStageSlots] = tau_t;
                sl[10 * kStageSlots] = __uint_as_float(cellp); sl[11 * kStageSlots] = __uint_as_float(meta);
                sl[12 * kStageSlots] = __uint_as_float(pkt); sl[13 * kStageSlots] = __uint_as_float(m_new);
            }
            staged += __popc(m_s);
            GCMCRT_CHECK(staged <= kStageSlots);
            __syncwarp();
        }
        // ---------------- phase 2: full warps of survivors start their flights; phase 3: long flights ----------------
        for (;;) {
            const bool do_long = in_flight >= 32 || (!more && staged == 0 && in_flight > 0);
            const bool do_new = !do_long && (staged >= 32 || (!more && staged > 0));
            if (!do_long && !do_new) break;
            const int n_take = min(do_long ? in_flight : staged, 32);
            const bool active = lane_id() < n_take;
            Ray ray{};
            float tau = 0.f, tau_t = 0.f, W = 0.f;
            uint32_t chan_run = 0, pkt = 0, m_new = 0;
            int st = RAY_NONE, used = 0;
            const float* alpha_c = rc.alpha;
            if (do_long) {
                if (active) flight_load(flights + (in_flight - n_take) + lane_id(), rc, gs, ray, tau, tau_t, W, chan_run, pkt,
                                        m_new, st, used, alpha_c);
                __syncwarp();
                in_flight -= n_take;
            } else {
                if (active) {
                    const float* sl = stage + (staged - n_take) + lane_id();
                    const float px = sl[0 * kStageSlots], py = sl[1 * kStageSlots], pz = sl[2 * kStageSlots];
                    W = sl[3 * kStageSlots];
                    float nx = sl[4 * kStageSlots], ny = sl[5 * kStageSlots], nz = sl[6 * kStageSlots];
                    const float ct = sl[7 * kStageSlots], zpsi = sl[8 * kStageSlots];
                    tau_t = sl[9 * kStageSlots];
                    const uint32_t cellp = __float_as_uint(sl[10 * kStageSlots]), meta = __float_as_uint(sl[11 * kStageSlots]);
                    pkt = __float_as_uint(sl[12 * kStageSlots]); m_new = __float_as_uint(sl[13 * kStageSlots]);
                    const uint32_t kind = meta & 3u;
                    chan_run = meta >> 8;
                    int i, j, k;
                    unpack_cell(cellp, i, j, k);
                    if (kind == EV_EMIT) {   // isotropic emission direction (Eq. 2), as the persistent kernel writes it
                        const float ns = sqrtf(fmaxf(0.f, 1.0f - ct * ct));
                        float sp, cp;
                        sincospif(2.0f * zpsi, &sp, &cp);
                        nx = ns * cp; ny = ns * sp; nz = ct;
                    } else {
                        rotate_dir(nx, ny, nz, ct, zpsi);   // about the incoming direction, or the surface normal (Eq. 4)
                        if (kind == EV_SURFACE) i = 0;
                    }
                    alpha_c = rc.alpha + (size_t)(rc.chan_begin + int(chan_run)) * rc.geom.alpha_stride;
                    ray_init(ray, gs, px, py, pz, nx, ny, nz, i, j, k, alpha_c);
                    if (!(FORCED && force_flight(rc, gs, ray, alpha_c, tau_t, W, wcnt.escw))) tau_t *= rc.inv_stretch;   // Sect. 4.2
                    st = RAY_FLYING;
                }
                __syncwarp();
                staged -= n_take;
            }
            used += wave_march<KSTEPS>(rc, gs, st, ray, tau, tau_t, alpha_c, do_long ? kLongRoundSteps : kFirstRoundSteps, wcnt);
            bool unfinished = active && (st == RAY_FLYING || st == RAY_PARK);
            if (unfinished && used > rc.geom.maxseg) { st = RAY_STUCK; unfinished = false; }
            wave_close(rc, ev, susp, wc.park_all, active && !unfinished, st, ray, W, tau, chan_run, pkt, m_new, wcnt);
            const unsigned m_u = __ballot_sync(kFullMask, unfinished);
            if (unfinished) flight_save(flights + in_flight + rank_in_mask(m_u), ray, tau, tau_t, W, chan_run, pkt, m_new, st, used);
            in_flight += __popc(m_u);
            GCMCRT_CHECK(in_flight <= kStageSlots && in_flight >= 0 && staged >= 0);
            __syncwarp();
        }
        if (!more) break;
    }
    wave_flush_counters(rc, wcnt);
}

}  // namespace gcmcrt

// gcmcrt.cu -- host side of libgcmcrt.so: the C-ABI of include/gcmcrt.h.
// Argument marshalling, device-memory ownership, kernel launches and the pass loop; all arithmetic of the method
// lives in kernels.cuh / ray.cuh / device_common.cuh.
#include "../../include/gcmcrt.h"

#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>
#include <string>
#include <vector>

#include "kernels.cuh"

using namespace gcmcrt;

namespace {

thread_local std::string g_create_error = "no error";

struct DevBuf {  // owned device allocation
    void* p = nullptr;
    size_t bytes = 0;
    void release() { if (p) cudaFree(p); p = nullptr; bytes = 0; }
    cudaError_t ensure(size_t n)
    {
        if (n <= bytes) return cudaSuccess;
        release();
        cudaError_t e = cudaMalloc(&p, n);
        if (e == cudaSuccess) bytes = n; else p = nullptr;
        return e;
    }
    template <class T> T* as() const { return static_cast<T*>(p); }
};

}  // namespace

struct gcmcrt_grid {
    int nlev = 0, nlat = 0, nlon = 0, ncell = 0;
    std::vector<double> r, th, ph;
    double Omega = 0.0;
    float surface_albedo = 0.f;
    int sm_count = 148;
    std::string err = "no error";

    // geometry + fields
    DevBuf tab, r64, cth64, ph64, rc32, thc32, phc32, T, rho, u, v, w;
    int tab_floats = 0;
    bool has_wind = false;

    // current opacity table
    int chan0 = 0, n_chan = 0;
    std::vector<float> lambda;
    std::vector<double> lambda64_h;
    std::vector<float> reff_h;
    DevBuf own_kabs, own_kray, own_kcld, own_g;   // copies of host-resident inputs
    const float *k_abs = nullptr, *k_ray = nullptr, *k_cld = nullptr, *g_cld = nullptr;
    DevBuf alpha, alpha2, prop, reff, vlos, lambda64;
    bool staged_cont = false;   // the staged tables are those of a continuous-absorption run (pair table, omega = 1)
    DevBuf node, node_idx, node_w, own_pcell;     // k_abs from (T, log10 p) node tables (gcmcrt_set_opacity_nodes)
    int nT = 0, nP = 0;
    std::vector<float> T_nodes_h, logp_nodes_h;
    bool use_nodes = false;
    int staged_obs = -2;   // -2: no tables set, -3: tables set but nothing staged yet (the first run stages what it needs),
                           // -1: unshifted table staged, >= 0: Doppler table of staged_dir staged
    double staged_dir[3] = {0, 0, 0};
    int staged_halfwidth = 0;
    int staged_c0 = 0, staged_c1 = 0;   // channels the staged tables hold (the whole table unless a part of a run staged them)

    // emission
    DevBuf Lcell, Lcum, Lcol, Ltot, guide;

    // workspace
    DevBuf ev0, evkeys, perm, hist, tile_sums, lkeys, lperm, lhist, ltile, flights, s0[2], s1[2], s2[2], ctrl, counters, counters_out, flux, ltot_out, value, sigma, image, evcount, contrib;
    unsigned int ev_cap = 0, ev_cap_forced = 0;
    bool tuned = false;   // environment overrides read
    int n_threads_resident = 0;
    // GCMCRT_TUNE="service,lateral,gens,batch_div": lanes waiting before the persistent kernel serves them; lanes parked at
    // a cone / half-plane before a warp serves them; wavefront generations per pass before the persistent kernel takes over
    // (0 = persistent kernel only); first-pass batch = event capacity / batch_div
    int tune[4] = {16, 1, 8, 4};
    PassCtrl* h_ctrl = nullptr;  // pinned (timed runs read the pass outcome back)
    cudaStream_t cap_stream = nullptr;   // the body of the pass loop is captured on this stream into the WHILE node's graph
    // instantiated pass-loop graphs, keyed by the bytes of everything their kernels were captured with: a repeated run
    // relaunches its graph, a run that differs in parameters only (other channels, observers, buffers) updates a graph of
    // the same shape in place (cudaGraphExecUpdate: microseconds, no allocation; launches already enqueued keep the old
    // parameters), and only a new shape (emission / albedo, generations, with or without peel-off) is instantiated.
    // cudaGraphExecDestroy waits for the device, so graphs pushed out of the cache are released at the library's next wait.
    struct LoopGraph { std::vector<unsigned char> key; unsigned shape = 0; cudaGraphExec_t exec = nullptr; cudaEvent_t done = nullptr; };
    std::vector<LoopGraph> loops, retired;
    cudaEvent_t tev[4] = {nullptr, nullptr, nullptr, nullptr};   // kernel timing (A0 | A2 | transport | peel)
    unsigned long long launches = 0, launches_pending = 0;
    double ms_stage = 0.0, ms_emis = 0.0, ms_transport = 0.0, ms_peel = 0.0, ms_sort = 0.0;
    double ms_stage_pending = 0.0;   // staging done by set_opacity, reported by the next run

    // run_params.concurrency: internal handles (grid copies with working buffers of their own) and the streams their parts of
    // a run are enqueued on; the opacity tables they borrow from this handle follow opacity_epoch
    std::vector<gcmcrt_grid*> peers;
    std::vector<cudaStream_t> peer_streams;
    std::vector<cudaEvent_t> peer_done;
    cudaEvent_t fork_ev = nullptr;
    DevBuf part_counters;
    unsigned long long opacity_epoch = 0, synced_epoch = 0;   // synced_epoch: on an internal handle, the owner's epoch its tables are from
    bool is_peer = false;
    const gcmcrt_grid* owner = nullptr;   // internal handle: the handle whose tables it borrows
};

namespace {

int fail(gcmcrt_grid* g, int code, const std::string& msg)
{
    if (g) g->err = msg; else g_create_error = msg;
    return code;
}

#define CUDA_TRY(g, expr)                                                                                 \
    do {                                                                                                  \
        cudaError_t e__ = (expr);                                                                         \
        if (e__ != cudaSuccess)                                                                           \
            return fail(g, e__ == cudaErrorMemoryAllocation ? GCMCRT_E_NOMEM : GCMCRT_E_CUDA,             \
                        std::string(#expr) + ": " + cudaGetErrorString(e__));                             \
    } while (0)

bool is_device_ptr(const void* p)
{
    cudaPointerAttributes a;
    if (cudaPointerGetAttributes(&a, p) != cudaSuccess) { cudaGetLastError(); return false; }
    return a.type == cudaMemoryTypeDevice || a.type == cudaMemoryTypeManaged;
}

// Return a device view of `src` (n elements): the pointer itself when it is device memory, else a copy in `own`.
template <class T>
cudaError_t device_view(const T* src, size_t n, DevBuf& own, cudaStream_t s, const T** out, bool force_copy = false)
{
    if (!src) { *out = nullptr; return cudaSuccess; }
    const bool dev = is_device_ptr(src);
    if (dev && !force_copy) { *out = src; return cudaSuccess; }
    cudaError_t e = own.ensure(n * sizeof(T));
    if (e != cudaSuccess) return e;
    e = cudaMemcpyAsync(own.p, src, n * sizeof(T), dev ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, s);
    *out = own.as<T>();
    return e;
}

template <class T>
cudaError_t upload(DevBuf& b, const std::vector<T>& v, cudaStream_t s)
{
    cudaError_t e = b.ensure(v.size() * sizeof(T));
    if (e != cudaSuccess) return e;
    return cudaMemcpyAsync(b.p, v.data(), v.size() * sizeof(T), cudaMemcpyHostToDevice, s);
}

GeomParams geom_params(const gcmcrt_grid* g)
{
    GeomParams gp;
    gp.nlev = g->nlev; gp.nlat = g->nlat; gp.nlon = g->nlon; gp.ncell = g->ncell;
    gp.tab = g->tab.as<float>();
    gp.tab_floats = g->tab_floats;
    gp.Rtoa = float(g->r[g->nlev]);
    gp.R0 = float(g->r[0]);
    gp.maxseg = 8 * (g->nlev + g->nlat + g->nlon) + 64;
    gp.col_stride = alpha_col_stride(g->nlev);
    gp.alpha_stride = (long long)g->nlat * g->nlon * gp.col_stride;
    return gp;
}

// floor(2^64 / d) for the kernels' exact division by a run constant (2^64 - 1 for d = 1)
unsigned long long magic_div(unsigned long long d)
{
    if (d <= 1) return ~0ull;
    return (unsigned long long)((((unsigned __int128)1) << 64) / d);
}

void normalize3(const double* in, float* out)
{
    const double n = std::sqrt(in[0] * in[0] + in[1] * in[1] + in[2] * in[2]);
    for (int m = 0; m < 3; ++m) out[m] = float(in[m] / (n > 0 ? n : 1.0));
}

// basis (e1, e2) perpendicular to unit d: e1 = normalize(z^ x d) (x^ if degenerate), e2 = d x e1   (O3, C19)
void perp_basis(const double* d, float* e1, float* e2)
{
    double a[3] = {-d[1], d[0], 0.0};
    const double n = std::sqrt(a[0] * a[0] + a[1] * a[1]);
    if (n < 1e-6) { a[0] = 1.0; a[1] = 0.0; a[2] = 0.0; } else { a[0] /= n; a[1] /= n; }
    const double b[3] = {d[1] * a[2] - d[2] * a[1], d[2] * a[0] - d[0] * a[2], d[0] * a[1] - d[1] * a[0]};
    for (int m = 0; m < 3; ++m) { e1[m] = float(a[m]); e2[m] = float(b[m]); }
}

cudaError_t ensure_events(gcmcrt_grid* g)
{
    for (auto& e : g->tev)
        if (!e) { cudaError_t r = cudaEventCreate(&e); if (r != cudaSuccess) return r; }
    return cudaSuccess;
}

// Stage alpha / prop for observer `obs_dir` (nullptr = unshifted table).
// c0 .. c1: the channels to stage (c1 = 0: the whole table)
int stage_opacity(gcmcrt_grid* g, const double* obs_dir, int halfwidth, cudaStream_t s, bool cont = false, bool timed = false,
                  int c0 = 0, int c1 = 0)
{
    if (c1 <= c0) { c0 = 0; c1 = g->n_chan; }
    const size_t n = size_t(g->n_chan) * g->ncell;
    const GeomParams gp0 = geom_params(g);
    const size_t n_alpha = size_t(g->n_chan) * size_t(gp0.alpha_stride);
    if (n_alpha * sizeof(float) > g->alpha.bytes) {
        // guard entries and padding are zero; the stage kernel writes the level entries only, and the layout of a
        // channel does not depend on n_chan, so the table is cleared once per allocation
        CUDA_TRY(g, g->alpha.ensure(n_alpha * sizeof(float)));
        CUDA_TRY(g, cudaMemsetAsync(g->alpha.p, 0, g->alpha.bytes, s));
    }
    if (cont && 2 * n_alpha * sizeof(float) > g->alpha2.bytes) {
        CUDA_TRY(g, g->alpha2.ensure(2 * n_alpha * sizeof(float)));
        CUDA_TRY(g, cudaMemsetAsync(g->alpha2.p, 0, g->alpha2.bytes, s));
    }
    CUDA_TRY(g, g->prop.ensure(n * sizeof(float4)));
    StageParams sp;
    sp.n_chan = g->n_chan; sp.ncell = g->ncell; sp.nlev = g->nlev; sp.nlat = g->nlat; sp.nlon = g->nlon;
    sp.c_begin = c0; sp.c_end = c1;
    sp.k_abs = g->k_abs; sp.k_ray = g->k_ray; sp.k_cld = g->k_cld; sp.g_cld = g->g_cld;
    sp.node = g->use_nodes ? g->node.as<float>() : nullptr;
    sp.node_idx = g->node_idx.as<int2>(); sp.node_w = g->node_w.as<float2>(); sp.nT = g->nT; sp.nP = g->nP;
    sp.rho = g->rho.as<float>();
    sp.alpha = g->alpha.as<float>(); sp.prop = g->prop.as<float4>();
    sp.alpha2 = cont ? g->alpha2.as<float>() : nullptr;
    sp.alpha_stride = gp0.alpha_stride; sp.col_stride = gp0.col_stride;
    sp.doppler = obs_dir != nullptr; sp.halfwidth = halfwidth;
    sp.vlos = nullptr; sp.reff = g->reff.as<float>();
    if (timed) {
        CUDA_TRY(g, ensure_events(g));
        CUDA_TRY(g, cudaEventRecord(g->tev[0], s));
    }
    if (obs_dir) {
        CUDA_TRY(g, g->vlos.ensure(size_t(g->ncell) * sizeof(float)));
        float o[3];
        normalize3(obs_dir, o);
        vlos_kernel<<<(g->ncell + 255) / 256, 256, 0, s>>>(g->nlev, g->nlat, g->nlon, g->u.as<float>(), g->v.as<float>(),
                                                          g->w.as<float>(), float(g->Omega), g->rc32.as<float>(),
                                                          g->thc32.as<float>(), g->phc32.as<float>(), o[0], o[1], o[2],
                                                          g->vlos.as<float>());
        sp.vlos = g->vlos.as<float>();
        ++g->launches;
    }
    {   // grid = (cell tiles, channel slices): every thread stages its cell for the channels of its slice
        const unsigned tiles = (unsigned)((g->ncell + 255) / 256);
        const unsigned want = (unsigned)std::max(1, g->sm_count * 16 / (int)std::max(1u, tiles));
        const unsigned slices = (unsigned)std::min<long long>(std::min<long long>((c1 - c0 + 3) / 4, 65535), std::max<long long>(want, 1));
        stage_kernel<<<dim3(tiles, slices), 256, 0, s>>>(sp);
    }
    CUDA_TRY(g, cudaGetLastError());
    ++g->launches;
    if (timed) {
        CUDA_TRY(g, cudaEventRecord(g->tev[1], s));
        CUDA_TRY(g, cudaEventSynchronize(g->tev[1]));
        float ms = 0.f;
        CUDA_TRY(g, cudaEventElapsedTime(&ms, g->tev[0], g->tev[1]));
        g->ms_stage_pending += ms;
    }
    g->staged_obs = obs_dir ? 0 : -1;
    g->staged_cont = cont;
    g->staged_c0 = c0; g->staged_c1 = c1;
    if (obs_dir) { for (int m = 0; m < 3; ++m) g->staged_dir[m] = obs_dir[m]; g->staged_halfwidth = halfwidth; }
    return GCMCRT_OK;
}

// Event buffer capacity: GCMCRT_EVENT_CAP if set (tests force tiny buffers with it); else what the run can use --
// about 4 events per packet -- between 1 Mi and 128 Mi events (128 Mi x 64 B = 8.6 GB of records plus 13 GB of
// parked-packet lists and sort arrays: a cfg2 step then takes 4 passes; 64 Mi / 7 passes measured 1.2 % slower).
// The buffers only ever grow.
int ensure_workspace(gcmcrt_grid* g, unsigned long long run_packets)
{
    if (!g->tuned) {
        g->tuned = true;
        if (const char* e = std::getenv("GCMCRT_EVENT_CAP")) {
            unsigned long long cap = std::strtoull(e, nullptr, 10);
            g->ev_cap_forced = (unsigned int)std::min<unsigned long long>(std::max<unsigned long long>(cap, 64), 1ull << 30);
        }
        if (const char* e = std::getenv("GCMCRT_TUNE")) {   // "service,lateral,generations,batch_div"
            int a = 0, b = 0, c = 0, d = 0;
            const int n = std::sscanf(e, "%d,%d,%d,%d", &a, &b, &c, &d);
            if (n >= 2) { g->tune[0] = std::min(std::max(a, 1), 32); g->tune[1] = std::min(std::max(b, 1), 32); }
            if (n >= 3) g->tune[2] = std::min(std::max(c, 0), kMaxGen);
            if (n >= 4) g->tune[3] = std::min(std::max(d, 1), 64);
        }
    }
    if (g->ev_cap_forced) {
        g->ev_cap = g->ev_cap_forced;
    } else {
        unsigned long long want = 1ull << 20;
        while (want < (128ull << 20) && want < 4 * run_packets) want <<= 1;
        if (want > g->ev_cap) g->ev_cap = (unsigned int)want;
    }
    CUDA_TRY(g, g->ev0.ensure(size_t(g->ev_cap) * 4 * sizeof(float4)));   // 64-byte records
    CUDA_TRY(g, g->perm.ensure(size_t(g->ev_cap) * sizeof(unsigned int)));
    CUDA_TRY(g, g->evkeys.ensure(size_t(g->ev_cap) * sizeof(unsigned int)));
    CUDA_TRY(g, g->ctrl.ensure(sizeof(PassCtrl)));
    CUDA_TRY(g, g->counters.ensure(sizeof(DevCounters)));
    if (!g->h_ctrl) CUDA_TRY(g, cudaMallocHost((void**)&g->h_ctrl, sizeof(PassCtrl)));
    return GCMCRT_OK;
}

struct OutBuf {  // an output array: the caller's device pointer, or an internal one copied back at the end
    void* dev = nullptr;
    void* host = nullptr;
    size_t bytes = 0;
};

int bind_out(gcmcrt_grid* g, void* user, size_t bytes, DevBuf& own, OutBuf& ob, bool always_internal = false)
{
    ob.bytes = bytes;
    if (user && is_device_ptr(user) && !always_internal) { ob.dev = user; ob.host = nullptr; return GCMCRT_OK; }
    CUDA_TRY(g, own.ensure(bytes > 0 ? bytes : 8));
    ob.dev = own.p;
    ob.host = (user && !is_device_ptr(user)) ? user : nullptr;
    return GCMCRT_OK;
}

// Everything one pass launches.  It is the same for every pass of a run: what changes from pass to pass (fresh packet
// range, which suspended list is read, the sort key window, the counters) lives in PassCtrl on the device.
struct PassLaunch {
    RunConst rc;
    EventBuf ev;
    SuspPair susp;
    WaveConst wc;
    SortParams sp, spl;
    PassPlan plan;
    PassCtrl* ctrl;
    int emission, has_obs;
    int n_gen, n_gen_run;
    unsigned grid_t, grid_f, grid_i, grid_p, grid_k;
    size_t smem_t, smem_w, smem_i, smem_p;
    decltype(&transport_kernel<4, false>) tk;
    decltype(&peel_kernel<16, false>) pk;
    decltype(&wave_first_flight_kernel<16, false>) k_first;
    decltype(&wave_interact_kernel<kInteractK, false>) k_inter;
    unsigned long long tail_items;
};   // zero-filled with memset before use: its bytes are the key of the graph cache

// kernels one pass launches (what enqueue_pass counts)
unsigned launches_per_pass(const PassLaunch& L)
{
    unsigned nl = 3;   // pass_begin, the persistent transport kernel, pass_end
    if (L.n_gen > 0) nl += (L.emission ? 1u : 6u) + unsigned(L.n_gen_run);
    if (L.has_obs) nl += 5u + (L.ev.hist ? 0u : 1u);
    return nl;
}

// Enqueue one pass on `s` (the caller's stream in a timed run, the capture stream of the loop body otherwise).
// tev != NULL: cudaEvents around the transport side, the event sort and the peel kernel.
int enqueue_pass(gcmcrt_grid* g, const PassLaunch& L, cudaStream_t s, cudaEvent_t* tev, cudaGraphConditionalHandle handle,
                 int use_handle, unsigned* n_launch)
{
    unsigned nl = 0;
    PassCtrl* ctrl = L.ctrl;
    pass_begin_kernel<<<1, 1, 0, s>>>(ctrl, L.plan);
    ++nl;
    if (tev) CUDA_TRY(g, cudaEventRecord(tev[0], s));
    // the event sort's histogram is filled while the records are written
    if (L.has_obs) CUDA_TRY(g, cudaMemsetAsync(L.sp.hist, 0, size_t(L.sp.nbins) * sizeof(unsigned int), s));
    if (L.n_gen > 0) {
        WaveConst wc = L.wc;
        if (!L.emission) {
            // launch-order sort of the fresh packets, then their first flights
            CUDA_TRY(g, cudaMemsetAsync(L.spl.hist, 0, size_t(L.spl.nbins) * sizeof(unsigned int), s));
            wave_launch_keys_kernel<<<L.grid_k, kWaveThreads, L.smem_w, s>>>(L.rc, wc);
            scan_reduce_kernel<<<L.spl.n_tiles, kScanThreads, 0, s>>>(L.spl);
            scan_tiles_kernel<<<1, 1024, 0, s>>>(L.spl);
            scan_apply_kernel<<<L.spl.n_tiles, kScanThreads, 0, s>>>(L.spl);
            ev_scatter_kernel<<<L.grid_k, 256, 0, s>>>(L.spl);
            L.k_first<<<L.grid_f, kWaveThreads, L.smem_w, s>>>(L.rc, L.ev, L.susp, wc);
            nl += 6;
        } else {
            wave_emit_kernel<<<L.grid_k, kWaveThreads, L.smem_w, s>>>(L.rc, L.ev, L.susp, wc);
            nl += 1;
        }
        gen_mark_kernel<<<1, 1, 0, s>>>(ctrl, 1);
        for (int gi = 0; gi < L.n_gen_run; ++gi) {
            wc.gen_mark = &ctrl->gen_mark[gi];
            wc.park_all = gi == L.n_gen - 1;
            L.k_inter<<<L.grid_i, kWaveThreads, L.smem_i, s>>>(L.rc, L.ev, L.susp, wc);
            gen_mark_kernel<<<1, 1, 0, s>>>(ctrl, gi + 2);
        }
        nl += unsigned(L.n_gen_run);
    }
    L.tk<<<L.grid_t, kTransportThreads, L.smem_t, s>>>(L.rc, L.ev, L.susp, L.tail_items);
    ++nl;
    if (tev) CUDA_TRY(g, cudaEventRecord(tev[1], s));
    if (L.has_obs) {
        // counting sort of this pass's events by (channel, cell): sort.cuh
        if (!L.ev.hist) { ev_hist_kernel<<<g->sm_count * 8, 256, 0, s>>>(L.sp); ++nl; }
        scan_reduce_kernel<<<L.sp.n_tiles, kScanThreads, 0, s>>>(L.sp);
        scan_tiles_kernel<<<1, 1024, 0, s>>>(L.sp);
        scan_apply_kernel<<<L.sp.n_tiles, kScanThreads, 0, s>>>(L.sp);
        ev_scatter_kernel<<<g->sm_count * 8, 256, 0, s>>>(L.sp);
        nl += 4;
    }
    if (tev) CUDA_TRY(g, cudaEventRecord(tev[2], s));
    if (L.has_obs) { L.pk<<<L.grid_p, kPeelThreads, L.smem_p, s>>>(L.rc, L.ev, L.sp.perm); ++nl; }
    if (tev) CUDA_TRY(g, cudaEventRecord(tev[3], s));
    pass_end_kernel<<<1, 1, 0, s>>>(ctrl, L.plan, handle, use_handle);
    ++nl;
    CUDA_TRY(g, cudaGetLastError());
    if (n_launch) *n_launch = nl;
    return GCMCRT_OK;
}

// The pass loop as a conditional WHILE node: the body is one pass, captured from enqueue_pass(); pass_end_kernel sets
// the condition.  Nothing here waits for the device.  When the caller's stream is itself being captured the node is
// added to the caller's graph (a graph that holds a conditional node cannot be a child graph); otherwise a graph of its
// own is instantiated, launched on the caller's stream and released (an executable graph in flight is freed on completion).
// cudaGraphExecDestroy waits for the device (measured: for as long as whatever is in flight takes, even when the graph
// itself has finished), so retired graphs are only released where the library waits anyway -- after the final
// synchronisation of a run with host outputs, in a timed run, in gcmcrt_destroy -- or when more than 256 have piled up.
void reap_retired_loops(gcmcrt_grid* g)
{
    for (auto& lg : g->retired) {
        cudaEventSynchronize(lg.done);
        cudaGraphExecDestroy(lg.exec);
        cudaEventDestroy(lg.done);
    }
    g->retired.clear();
    cudaGetLastError();
}

int launch_pass_loop(gcmcrt_grid* g, const PassLaunch& L, cudaStream_t s, unsigned* n_launch)
{
    constexpr size_t kLoopCache = 8;
    const unsigned shape = 1u | (L.emission ? 2u : 0u) | (L.has_obs ? 4u : 0u) | (L.ev.hist ? 8u : 0u) | unsigned(L.n_gen) << 4 |
                           unsigned(L.n_gen_run) << 12;
    if (!g->cap_stream) CUDA_TRY(g, cudaStreamCreateWithFlags(&g->cap_stream, cudaStreamNonBlocking));
    cudaStreamCaptureStatus cst = cudaStreamCaptureStatusNone;
    CUDA_TRY(g, cudaStreamIsCapturing(s, &cst));
    cudaGraph_t graph = nullptr;
    const cudaGraphNode_t* deps = nullptr;
    size_t n_deps = 0;
    const bool own = cst != cudaStreamCaptureStatusActive;
    const unsigned char* kb = reinterpret_cast<const unsigned char*>(&L);
    if (own) {
        if (g->retired.size() > 256) reap_retired_loops(g);
        for (size_t m = 0; m < g->loops.size(); ++m) {
            if (g->loops[m].key.size() == sizeof L && std::memcmp(g->loops[m].key.data(), kb, sizeof L) == 0) {
                gcmcrt_grid::LoopGraph lg = g->loops[m];   // most recently used goes to the back
                g->loops.erase(g->loops.begin() + m);
                g->loops.push_back(lg);
                if (n_launch) *n_launch = launches_per_pass(L);
                CUDA_TRY(g, cudaGraphLaunch(lg.exec, s));
                CUDA_TRY(g, cudaEventRecord(lg.done, s));
                return GCMCRT_OK;
            }
        }
        CUDA_TRY(g, cudaGraphCreate(&graph, 0));
    } else {
        unsigned long long id = 0;
        CUDA_TRY(g, cudaStreamGetCaptureInfo(s, &cst, &id, &graph, &deps, &n_deps));
    }
    int rcode = GCMCRT_OK;
    cudaGraphNode_t node = nullptr;
    do {
        cudaGraphConditionalHandle handle;
        cudaError_t e = cudaGraphConditionalHandleCreate(&handle, graph, 1, cudaGraphCondAssignDefault);
        cudaGraphNodeParams np = {};
        np.type = cudaGraphNodeTypeConditional;
        np.conditional.handle = handle;
        np.conditional.type = cudaGraphCondTypeWhile;
        np.conditional.size = 1;
        if (e == cudaSuccess) e = cudaGraphAddNode(&node, graph, deps, n_deps, &np);
        if (e == cudaSuccess) e = cudaStreamBeginCaptureToGraph(g->cap_stream, np.conditional.phGraph_out[0], nullptr, nullptr, 0,
                                                               cudaStreamCaptureModeRelaxed);
        if (e != cudaSuccess) { rcode = fail(g, GCMCRT_E_CUDA, std::string("pass loop graph: ") + cudaGetErrorString(e)); break; }
        rcode = enqueue_pass(g, L, g->cap_stream, nullptr, handle, 1, n_launch);
        cudaGraph_t body = nullptr;
        e = cudaStreamEndCapture(g->cap_stream, &body);
        if (rcode == GCMCRT_OK && e != cudaSuccess) rcode = fail(g, GCMCRT_E_CUDA, std::string("pass loop capture: ") + cudaGetErrorString(e));
        if (rcode != GCMCRT_OK) break;
        if (own) {
            // a cached graph of the same shape takes the new parameters in place
            bool updated = false;
            for (size_t m = g->loops.size(); m-- > 0 && !updated;) {
                if (g->loops[m].shape != shape) continue;
                cudaGraphExecUpdateResultInfo info;
                if (cudaGraphExecUpdate(g->loops[m].exec, graph, &info) == cudaSuccess && info.result == cudaGraphExecUpdateSuccess) {
                    gcmcrt_grid::LoopGraph lg = g->loops[m];
                    g->loops.erase(g->loops.begin() + m);
                    lg.key.assign(kb, kb + sizeof L);
                    e = cudaGraphLaunch(lg.exec, s);
                    if (e == cudaSuccess) e = cudaEventRecord(lg.done, s);
                    g->loops.push_back(lg);
                    updated = true;
                } else {
                    cudaGetLastError();
                    break;   // same shape but not updatable (a memset outgrew its node): instantiate
                }
            }
            if (updated) {
                if (e != cudaSuccess) rcode = fail(g, GCMCRT_E_CUDA, std::string("pass loop launch: ") + cudaGetErrorString(e));
                break;
            }
            gcmcrt_grid::LoopGraph lg;
            lg.shape = shape;
            e = cudaGraphInstantiate(&lg.exec, graph, 0);
            if (e == cudaSuccess) e = cudaEventCreateWithFlags(&lg.done, cudaEventDisableTiming);
            if (e == cudaSuccess) e = cudaGraphLaunch(lg.exec, s);
            if (e == cudaSuccess) e = cudaEventRecord(lg.done, s);
            if (e == cudaSuccess) {
                lg.key.assign(kb, kb + sizeof L);
                if (g->loops.size() >= kLoopCache) { g->retired.push_back(g->loops.front()); g->loops.erase(g->loops.begin()); }
                g->loops.push_back(lg);
            } else {
                if (lg.done) cudaEventDestroy(lg.done);
                if (lg.exec) cudaGraphExecDestroy(lg.exec);
            }
        } else {
            e = cudaStreamUpdateCaptureDependencies(s, &node, 1, cudaStreamSetCaptureDependencies);
        }
        if (e != cudaSuccess) rcode = fail(g, GCMCRT_E_CUDA, std::string("pass loop launch: ") + cudaGetErrorString(e));
    } while (0);
    if (own && graph) cudaGraphDestroy(graph);
    if (rcode != GCMCRT_OK) cudaGetLastError();
    return rcode;
}

// The counters of the ABI, assembled on the device (so that a run with device outputs needs no host round trip).
__global__ void finalize_counters_kernel(const DevCounters* dc, const PassCtrl* c, gcmcrt_counters* out, unsigned long long launches_fixed,
                                         unsigned long long launches_per_pass, unsigned long long passes_extra, double ms_stage,
                                         double ms_emis, double ms_transport, double ms_peel, double ms_sort)
{
    gcmcrt_counters hc;
    hc.events = dc->events; hc.segments_transport = dc->seg_transport; hc.segments_peel = dc->seg_peel;
    hc.packets_escaped = dc->escaped; hc.packets_absorbed = dc->absorbed; hc.packets_surface = dc->surface;
    hc.packets_stuck = dc->stuck; hc.escaped_weight = dc->escaped_weight; hc.rays_peel = dc->rays_peel;
    const unsigned long long passes = c ? c->passes : 0ull;
    hc.passes = passes + passes_extra;
    hc.launches = launches_fixed + launches_per_pass * passes;
    hc.ms_stage = ms_stage; hc.ms_emission_cdf = ms_emis; hc.ms_transport = ms_transport; hc.ms_peel = ms_peel; hc.ms_sort = ms_sort;
    hc.device_status = c ? (unsigned long long)c->error : 0ull;
    *out = hc;
}

// mode: 0 albedo, 1 emission, 2 transmission
// part: the call is one part of a run cut by run_split(): tables are staged, and the emission CDF is built, for the
// channels of the part only
int run_mode(gcmcrt_grid* g, const gcmcrt_run_params* prm, gcmcrt_result* out, void* stream, int mode, bool part = false)
{
    const int emission = mode == 1;
    if (!g) return GCMCRT_E_INVALID;
    if (!prm || !out) return fail(g, GCMCRT_E_INVALID, "params and result must not be NULL");
    if (g->n_chan <= 0 || g->staged_obs == -2) return fail(g, GCMCRT_E_STATE, "gcmcrt_set_opacity has not been called");
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    const int n_obs = prm->n_obs;
    if (n_obs < 0 || n_obs > kMaxObs) return fail(g, GCMCRT_E_INVALID, "n_obs must be in [0, 32]");
    if (n_obs > 0 && !prm->obs_dir) return fail(g, GCMCRT_E_INVALID, "obs_dir is NULL");
    const unsigned long long N = prm->packets_per_channel;
    if (N == 0 || N > 0xffffffffull) return fail(g, GCMCRT_E_INVALID, "packets_per_channel must be in [1, 2^32)");
    const unsigned long long lo = prm->pkt_begin, hi = prm->pkt_end ? prm->pkt_end : N;
    if (lo > hi || hi > N) return fail(g, GCMCRT_E_INVALID, "bad packet range");
    const int cb = prm->chan_begin, ce = prm->chan_end ? prm->chan_end : g->n_chan;
    if (cb < 0 || ce > g->n_chan || cb >= ce) return fail(g, GCMCRT_E_INVALID, "bad channel range");
    const int nb = prm->n_batches ? prm->n_batches : 32;
    if (nb < 1 || nb > kMaxBatches) return fail(g, GCMCRT_E_INVALID, "n_batches must be in [1, 64]");
    if (!out->flux_sum && n_obs > 0) return fail(g, GCMCRT_E_INVALID, "result.flux_sum is required");
    if (prm->emission_bias < 0.0 || prm->emission_bias >= 1.0) return fail(g, GCMCRT_E_INVALID, "emission_bias must be in [0,1)");
    if (prm->roulette_w_min < 0.0 || (prm->roulette_w_min > 0.0 && !(prm->roulette_survive > 0.0 && prm->roulette_survive <= 1.0)))
        return fail(g, GCMCRT_E_INVALID, "roulette: w_min >= 0 and 0 < survive <= 1 required");
    if (prm->roulette_w_min > 0.0 && !prm->survival_bias) return fail(g, GCMCRT_E_INVALID, "roulette requires survival_bias");
    if (prm->doppler_on && g->n_chan > 1 && g->reff.p == nullptr) return fail(g, GCMCRT_E_STATE, "no wavelength table");
    const int ncr = ce - cb;
    if (ncr > (1 << 24)) return fail(g, GCMCRT_E_INVALID, "too many channels in one run");
    const int npix = prm->npix > 0 && out->image ? prm->npix : 0;
    const bool timed = prm->timing != 0;   // host-synchronous pass loop with cudaEvents around the kernels
    // Sect. 5.1 with multiple scattering (L259, N12): after the chords' initial peel-off the packets are transported
    const bool ms_trans = mode == 2 && prm->scatter_on && prm->star_solid_angle > 0.0;
    // GCMCRT_HOST_LOOP=1: the host drives the pass loop (one wait per pass) without recording events -- for profilers,
    // which do not see kernels launched from inside a conditional graph node
    static const bool host_loop_env = std::getenv("GCMCRT_HOST_LOOP") && std::atoi(std::getenv("GCMCRT_HOST_LOOP")) != 0;

    int rcode = ensure_workspace(g, (unsigned long long)ncr * (hi - lo));
    if (rcode) return rcode;
    if (prm->forced_scatter < 0 || prm->forced_scatter > 2 || (prm->forced_scatter && prm->continuous_absorption))
        return fail(g, GCMCRT_E_INVALID, "forced_scatter must be 0, 1 or 2 and excludes continuous_absorption");
    if (prm->forced_scatter == 2 && !(prm->max_events > 0 || (prm->survival_bias && prm->roulette_w_min > 0.0)))
        return fail(g, GCMCRT_E_INVALID, "forced_scatter = 2 needs max_events or Russian roulette to end its packets");
    if (prm->cloud_phase < 0 || prm->cloud_phase > 2) return fail(g, GCMCRT_E_INVALID, "cloud_phase must be 0 (HG), 1 (TTHG) or 2 (Draine)");
    if (!(prm->stretch_alpha >= 0.0 && prm->stretch_alpha <= 1.0) || (prm->stretch_alpha > 0.0 && prm->stretch_alpha < 1.0 && prm->continuous_absorption))
        return fail(g, GCMCRT_E_INVALID, "stretch_alpha must be in [0, 1] and excludes continuous_absorption");
    if (mode == 2 && n_obs < 1) return fail(g, GCMCRT_E_INVALID, "transmission needs at least one observer direction");
    if (!(prm->star_solid_angle >= 0.0)) return fail(g, GCMCRT_E_INVALID, "star_solid_angle must be >= 0");

    // ---- outputs
    OutBuf o_flux, o_ltot, o_val, o_sig, o_img, o_evc, o_ctb, o_cnt;
    const size_t nflux = size_t(ncr) * std::max(n_obs, 1) * nb;
    if ((rcode = bind_out(g, out->flux_sum, nflux * sizeof(double), g->flux, o_flux))) return rcode;
    if ((rcode = bind_out(g, out->L_tot, size_t(ncr) * std::max(n_obs, 1) * sizeof(double), g->ltot_out, o_ltot))) return rcode;
    if ((rcode = bind_out(g, out->value, size_t(ncr) * std::max(n_obs, 1) * sizeof(double), g->value, o_val))) return rcode;
    if ((rcode = bind_out(g, out->sigma, size_t(ncr) * std::max(n_obs, 1) * sizeof(double), g->sigma, o_sig))) return rcode;
    if (npix) if ((rcode = bind_out(g, out->image, size_t(ncr) * n_obs * npix * npix * sizeof(float), g->image, o_img))) return rcode;
    const size_t n_pkt = size_t(hi - lo);
    if (out->event_count) if ((rcode = bind_out(g, out->event_count, size_t(ncr) * n_pkt * sizeof(uint32_t), g->evcount, o_evc))) return rcode;
    if (out->counters) if ((rcode = bind_out(g, out->counters, sizeof(gcmcrt_counters), g->counters_out, o_cnt))) return rcode;
    CUDA_TRY(g, cudaMemsetAsync(o_flux.dev, 0, nflux * sizeof(double), s));
    CUDA_TRY(g, cudaMemsetAsync(o_ltot.dev, 0, o_ltot.bytes, s));
    if (npix) CUDA_TRY(g, cudaMemsetAsync(o_img.dev, 0, o_img.bytes, s));
    if (out->contrib && n_obs > 0) {
        if ((rcode = bind_out(g, out->contrib, size_t(ncr) * n_obs * 2 * g->ncell * sizeof(float), g->contrib, o_ctb))) return rcode;
        CUDA_TRY(g, cudaMemsetAsync(o_ctb.dev, 0, o_ctb.bytes, s));
    }
    if (o_evc.dev) CUDA_TRY(g, cudaMemsetAsync(o_evc.dev, 0, o_evc.bytes, s));
    CUDA_TRY(g, cudaMemsetAsync(g->counters.p, 0, sizeof(DevCounters), s));

    // ---- constants of the run
    PassLaunch L;
    std::memset(static_cast<void*>(&L), 0, sizeof L);
    L.grid_t = L.grid_f = L.grid_i = L.grid_p = L.grid_k = 1;
    RunConst& rc = L.rc;
    rc.geom = geom_params(g);
    rc.chan_key0 = uint32_t(g->chan0);
    rc.chan_begin = cb; rc.n_chan_run = ncr;
    rc.pkt_begin = uint32_t(lo); rc.n_pkt = uint32_t(n_pkt);
    rc.N = N; rc.seed = prm->seed;
    rc.mode = emission;
    rc.max_events = prm->max_events; rc.scatter_on = prm->scatter_on;
    rc.survival_bias = prm->survival_bias != 0;
    rc.cloud_phase = prm->cloud_phase;
    rc.forced_scatter = prm->forced_scatter;
    rc.launch_chord = 0;
    rc.stretch = (prm->stretch_alpha > 0.0 && prm->stretch_alpha < 1.0) ? float(prm->stretch_alpha) : 1.0f;
    rc.inv_stretch = 1.0f / rc.stretch;
    rc.alpha2 = nullptr;
    rc.roulette_w_min = float(prm->roulette_w_min); rc.roulette_survive = float(prm->roulette_survive);
    rc.surface_albedo = g->surface_albedo;
    rc.xi = prm->emission_bias;
    rc.n_batches = nb;
    rc.n_obs_total = std::max(n_obs, 1);
    normalize3(prm->star_dir, rc.star);
    for (int m = 0; m < 3; ++m) rc.launch_dir[m] = -rc.star[m];
    {
        double sd[3] = {rc.star[0], rc.star[1], rc.star[2]};
        perp_basis(sd, rc.e1, rc.e2);
    }
    for (int o = 0; o < n_obs; ++o) {
        normalize3(prm->obs_dir + 3 * o, rc.obs[o]);
        double od[3] = {rc.obs[o][0], rc.obs[o][1], rc.obs[o][2]};
        perp_basis(od, rc.img_ex[o], rc.img_ey[o]);
    }
    rc.tau_cut = float(prm->tau_cut > 0.0 ? prm->tau_cut : 50.0);
    rc.npix = npix;
    rc.flux = static_cast<double*>(o_flux.dev);
    rc.image = npix ? static_cast<float*>(o_img.dev) : nullptr;
    rc.contrib = static_cast<float*>(o_ctb.dev);
    rc.event_count = static_cast<uint32_t*>(o_evc.dev);
    rc.counters = g->counters.as<DevCounters>();
    rc.magic_N = magic_div(N);
    rc.magic_npkt = magic_div(n_pkt);
    rc.t_service = g->tune[0]; rc.t_lateral = g->tune[1]; rc.p_refill = 12;
    PassCtrl* ctrl = g->ctrl.as<PassCtrl>();
    L.ctrl = ctrl;
    rc.work_counter = &ctrl->work_counter;
    rc.ray_counter = &ctrl->ray_counter;
    rc.ctrl = ctrl;

    // ---- launch geometry: persistent grids sized to the device
    const size_t smem_t = size_t(g->tab_floats) * sizeof(float);
    int occ_t = 0, occ_p = 0;
    const bool cont = prm->continuous_absorption != 0;
    L.tk = cont ? transport_kernel<4, true> : transport_kernel<4, false>;
    L.pk = peel_kernel<16, false>;
    L.emission = emission != 0 ? 1 : 0;
    L.smem_t = smem_t;
    if (mode != 2 || ms_trans) {
        CUDA_TRY(g, cudaFuncSetAttribute(L.tk, cudaFuncAttributeMaxDynamicSharedMemorySize, int(smem_t)));
        CUDA_TRY(g, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ_t, L.tk, kTransportThreads, smem_t));
        if (occ_t < 1) return fail(g, GCMCRT_E_INVALID, "grid tables do not fit in shared memory");
    }
    L.grid_t = unsigned(g->sm_count * std::max(occ_t, 1));
    const unsigned long long threads_t = (unsigned long long)L.grid_t * kTransportThreads;
    // suspended list: one entry per resident lane for the persistent kernel, plus what a wavefront pass can park (its
    // last generation and whatever found the event buffer full).  A pass starts with at most ev_cap / 2 inherited
    // entries (else it only drains) and parks each of its <= ev_cap / 2 fresh packets at most once: <= ev_cap in all
    const unsigned long long susp_cap = threads_t + (g->tune[2] > 0 ? 1ull * g->ev_cap : 0ull);
    if (mode != 2 || ms_trans) {
        for (int b = 0; b < 2; ++b) {
            CUDA_TRY(g, g->s0[b].ensure(susp_cap * sizeof(float4)));
            CUDA_TRY(g, g->s1[b].ensure(susp_cap * sizeof(float4)));
            CUDA_TRY(g, g->s2[b].ensure(susp_cap * sizeof(uint4)));
            SuspBuf& sb = L.susp.b[b];
            sb.s0 = g->s0[b].as<float4>(); sb.s1 = g->s1[b].as<float4>(); sb.s2 = g->s2[b].as<uint4>();
            sb.count = &ctrl->susp_count[b]; sb.taken = &ctrl->susp_taken[b];
            sb.cap = (unsigned int)std::min<unsigned long long>(susp_cap, 0xffffffffull);
        }
    }
    EventBuf& ev = L.ev;
    ev.rec = g->ev0.as<float4>();
    ev.count = &ctrl->ev_count;
    ev.cap = g->ev_cap;
    ev.soft_cap = (unsigned long long)g->ev_cap > 4 * threads_t ? g->ev_cap - (unsigned int)(2 * threads_t) : g->ev_cap / 2;
    ev.chan_lo = &ctrl->chan_lo;

    const int n_runs = (prm->doppler_on || ms_trans) ? std::max(n_obs, 1) : 1;   // one run per observer: its own table / its own chords
    unsigned long long passes_host = 0;   // transmission: one "pass" per run, counted here
    unsigned launches_per_pass = 0;
    if (timed) CUDA_TRY(g, ensure_events(g));
    g->launches = g->launches_pending; g->launches_pending = 0; g->ms_emis = g->ms_transport = g->ms_peel = g->ms_sort = 0.0;
    g->ms_stage = 0.0;
    CUDA_TRY(g, cudaMemsetAsync(ctrl, 0, sizeof(PassCtrl), s));
    const int st0 = part ? cb : 0, st1 = part ? ce : g->n_chan;   // channels whose staged tables and CDF this call needs
    for (int run = 0; run < n_runs; ++run) {
        // ---- A0/A1: make sure the staged table is the one this run needs
        if (prm->doppler_on && n_obs > 0) {
            const double* od = prm->obs_dir + 3 * run;
            const bool same = g->staged_obs >= 0 && g->staged_cont == cont && g->staged_halfwidth == prm->doppler_halfwidth &&
                              g->staged_dir[0] == od[0] && g->staged_dir[1] == od[1] && g->staged_dir[2] == od[2] &&
                              g->staged_c0 <= st0 && st1 <= g->staged_c1;
            if (!same && (rcode = stage_opacity(g, od, prm->doppler_halfwidth, s, cont, timed, st0, st1))) return rcode;
            rc.obs_first = run; rc.n_obs_run = 1;
        } else {
            if ((g->staged_obs != -1 || g->staged_cont != cont || g->staged_c0 > st0 || st1 > g->staged_c1) &&
                (rcode = stage_opacity(g, nullptr, 0, s, cont, timed, st0, st1))) return rcode;
            rc.obs_first = 0; rc.n_obs_run = n_obs;
            if (ms_trans) { rc.obs_first = run; rc.n_obs_run = 1; }
        }
        rc.magic_nobs = magic_div((unsigned long long)std::max(rc.n_obs_run, 1));
        rc.alpha = g->alpha.as<float>();
        rc.alpha2 = cont ? g->alpha2.as<float>() : nullptr;
        rc.prop = g->prop.as<float4>();
        // ---- A2: emission CDF
        if (emission) {
            const size_t n = size_t(g->n_chan) * g->ncell;
            if (prm->emission_bias > 0.0) CUDA_TRY(g, g->Lcell.ensure(n * sizeof(double)));
            CUDA_TRY(g, g->Lcum.ensure(n * sizeof(double)));
            CUDA_TRY(g, g->Lcol.ensure(size_t(g->n_chan) * g->nlat * g->nlon * sizeof(double)));
            CUDA_TRY(g, g->Ltot.ensure(size_t(g->n_chan) * sizeof(double)));
            EmisParams ep;
            ep.n_chan = g->n_chan; ep.nlev = g->nlev; ep.nlat = g->nlat; ep.nlon = g->nlon; ep.ncell = g->ncell;
            ep.alpha = rc.alpha; ep.prop = rc.prop;
            ep.alpha_stride = rc.geom.alpha_stride; ep.col_stride = rc.geom.col_stride;
            ep.rho = g->rho.as<float>(); ep.T = g->T.as<float>();
            ep.lambda = g->lambda64.as<double>();
            ep.r_edges = g->r64.as<double>(); ep.cth_edges = g->cth64.as<double>(); ep.ph_edges = g->ph64.as<double>();
            ep.tau_vert_max = prm->tau_vert_max;
            ep.Lcell = prm->emission_bias > 0.0 ? g->Lcell.as<double>() : nullptr; ep.Lcum = g->Lcum.as<double>(); ep.Lcol = g->Lcol.as<double>(); ep.Ltot = g->Ltot.as<double>();
            if (timed) CUDA_TRY(g, cudaEventRecord(g->tev[0], s));
            CUDA_TRY(g, g->guide.ensure(size_t(g->n_chan) * kEmisGuide * sizeof(int)));
            {
                // the CDF of the run's own channels cb .. ce (the tables are indexed by table channel): the same kernels
                // on pointers that start at channel cb.  blockIdx.y = channel; the warps of a channel's CTAs stride
                // through its columns
                const int ncol = g->nlat * g->nlon, wpb = kEmisThreads / 32;
                EmisParams er = ep;
                er.n_chan = ncr;
                er.alpha += size_t(cb) * er.alpha_stride; er.prop += size_t(cb) * g->ncell; er.lambda += cb;
                if (er.Lcell) er.Lcell += size_t(cb) * g->ncell;
                er.Lcum += size_t(cb) * g->ncell; er.Lcol += size_t(cb) * ncol; er.Ltot += cb;
                const dim3 ge((unsigned)std::min((ncol + wpb - 1) / wpb, 32), (unsigned)std::min(ncr, 65535));
                const size_t sm = 2 * size_t(g->nlev) * sizeof(double);
                if (g->nlev <= 64) emis_col_kernel<2><<<ge, kEmisThreads, sm, s>>>(er);
                else if (g->nlev <= 128) emis_col_kernel<4><<<ge, kEmisThreads, sm, s>>>(er);
                else if (g->nlev <= 256) emis_col_kernel<8><<<ge, kEmisThreads, sm, s>>>(er);
                else return fail(g, GCMCRT_E_INVALID, "emission: nlev > 256 is not supported");
                emis_colscan_kernel<<<(unsigned)((size_t(ncr) * 32 + 127) / 128), 128, 0, s>>>(ncr, ncol, er.Lcol, er.Ltot);
                emis_guide_kernel<<<(unsigned)(((long long)ncr * kEmisGuide + 255) / 256), 256, 0, s>>>(
                    ncr, g->ncell, g->nlev, er.Lcum, er.Lcol, er.Ltot, g->guide.as<int>() + size_t(cb) * kEmisGuide);
            }
            CUDA_TRY(g, cudaGetLastError());
            if (timed) {
                CUDA_TRY(g, cudaEventRecord(g->tev[1], s));
                CUDA_TRY(g, cudaEventSynchronize(g->tev[1]));
                float ms = 0.f;
                CUDA_TRY(g, cudaEventElapsedTime(&ms, g->tev[0], g->tev[1]));
                g->ms_emis += ms;
            }
            g->launches += 3;
            rc.Lcum = ep.Lcum; rc.Lcol = ep.Lcol; rc.Lcell = ep.Lcell; rc.Ltot = ep.Ltot; rc.guide = g->guide.as<int>();
            // L_tot output [n_chan_run][n_obs]
            const int o0 = prm->doppler_on ? run : 0, o1 = prm->doppler_on ? run + 1 : std::max(n_obs, 1);
            for (int o = o0; o < o1; ++o)
                CUDA_TRY(g, cudaMemcpy2DAsync(static_cast<double*>(o_ltot.dev) + o, sizeof(double) * rc.n_obs_total,
                                              ep.Ltot + cb, sizeof(double), sizeof(double), ncr,
                                              cudaMemcpyDeviceToDevice, s));
        }
        // event counts are recorded for the first run only (with doppler_on: observer 0's run)
        rc.event_count = run == 0 ? static_cast<uint32_t*>(o_evc.dev) : nullptr;

        const unsigned long long total_items = (unsigned long long)ncr * n_pkt;
        if (mode == 2) {
            // ---- transmission (Sect. 5.1): one chord per packet and observer, no events, no passes
            auto k_tr = transmission_kernel<8>;
            int occ_tr = 1;
            CUDA_TRY(g, cudaFuncSetAttribute(k_tr, cudaFuncAttributeMaxDynamicSharedMemorySize, int(smem_t)));
            CUDA_TRY(g, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ_tr, k_tr, 256, smem_t));
            if (occ_tr < 1) return fail(g, GCMCRT_E_INVALID, "grid tables do not fit in shared memory");
            if (timed) CUDA_TRY(g, cudaEventRecord(g->tev[2], s));
            for (int o = rc.obs_first; o < rc.obs_first + rc.n_obs_run; ++o) {
                TransParams tp;
                tp.o = o;
                for (int m = 0; m < 3; ++m) { tp.ex[m] = rc.img_ex[o][m]; tp.ey[m] = rc.img_ey[o][m]; }
                tp.star_radius = float(prm->star_radius);
                tp.planet_x = float(prm->planet_xy[0]); tp.planet_y = float(prm->planet_xy[1]);
                tp.ld_c1 = float(prm->ld_c1); tp.ld_c2 = float(prm->ld_c2);
                const unsigned gt = (unsigned)std::min<unsigned long long>((total_items + 255) / 256, (unsigned long long)g->sm_count * occ_tr);
                k_tr<<<std::max(gt, 1u), 256, smem_t, s>>>(rc, tp, total_items);
                ++g->launches;
            }
            CUDA_TRY(g, cudaGetLastError());
            if (timed) {
                CUDA_TRY(g, cudaEventRecord(g->tev[3], s));
                CUDA_TRY(g, cudaEventSynchronize(g->tev[3]));
                float c = 0.f;
                CUDA_TRY(g, cudaEventElapsedTime(&c, g->tev[2], g->tev[3]));
                g->ms_peel += c;
            }
            ++passes_host;
            if (!ms_trans) continue;
            // the packets go on from their chords' starts toward this run's observer; their peel-offs are taken off the
            // chords' terms by the peel kernel (chord_scale)
            const int o = rc.obs_first;
            rc.launch_chord = 1;
            for (int m = 0; m < 3; ++m) { rc.launch_dir[m] = rc.obs[o][m]; rc.tr_ex[m] = rc.img_ex[o][m]; rc.tr_ey[m] = rc.img_ey[o][m]; }
            rc.tr_star_radius = float(prm->star_radius);
            rc.tr_planet_x = float(prm->planet_xy[0]); rc.tr_planet_y = float(prm->planet_xy[1]);
            rc.tr_ld_c1 = float(prm->ld_c1); rc.tr_ld_c2 = float(prm->ld_c2);
            rc.tr_domega = float(prm->star_solid_angle);
        }

        // ---- the pass loop of this run
        L.has_obs = rc.n_obs_run > 0 ? 1 : 0;
        // several observers in one run: some lie below the horizon of most events, and the instance with the horizon test
        // does not set those rays up (cfg3: peel 174.4 -> 166.7 ms); with one observer the test costs more than it saves
        // (cfg2 +0.9 ms, cfg4 +0.7 ms, cfg5 +1.4 ms per 2048 wavelengths).  Same results either way.
        L.pk = rc.n_obs_run > 1 ? peel_kernel<16, true> : peel_kernel<16, false>;
        const size_t smem_p = (size_t((g->tab_floats + 31) & ~31) + size_t(kPeelThreads / 32) * rc.n_obs_run * nb) * sizeof(float);
        L.smem_p = smem_p;
        if (L.has_obs) {
            CUDA_TRY(g, cudaFuncSetAttribute(L.pk, cudaFuncAttributeMaxDynamicSharedMemorySize, int(smem_p)));
            CUDA_TRY(g, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ_p, L.pk, kPeelThreads, smem_p));
            if (occ_p < 1) return fail(g, GCMCRT_E_INVALID, "peel bins do not fit in shared memory");
            L.grid_p = unsigned(g->sm_count * occ_p);
        }
        SortParams& sp = L.sp;
        if (L.has_obs) {
            const long long max_bins = 1ll << 25;
            // channels whose events can share one pass: every packet makes at least one event when it interacts,
            // so a pass of ev_cap events spans about ev_cap / n_pkt channels; more bins than that only cost scan time
            const long long span = (long long)(g->ev_cap / std::max<size_t>(n_pkt, 1)) + 2;
            // few packets per channel (high-resolution runs: 1e5 packets over 1e5-1e6 cells): a coarser second key part
            // -- groups of 4 levels below 2 packets per cell, whole columns below 1 packet per 4 cells.  Rays from one
            // column toward one observer still share their extinction sectors, the histogram shrinks and every channel
            // of the pass keeps bins of its own; lanes of different levels finish at different steps, which costs the
            // peel kernel more than the smaller sort saves once the bins are well filled
            const int lev_shift = n_pkt >= 2ull * (unsigned long long)g->ncell ? 0 : (4 * n_pkt >= (unsigned long long)g->ncell ? 2 : 30);
            const long long nlg = lev_shift >= 30 ? 1 : (g->nlev + (1 << lev_shift) - 1) >> lev_shift;
            const long long bins_per_chan = (long long)g->nlat * g->nlon * nlg;
            sp.c_fold = int(std::max<long long>(1, std::min<long long>(std::min<long long>(ncr, max_bins / bins_per_chan), span)));
            sp.nbins = (unsigned int)((long long)sp.c_fold * bins_per_chan);
            ev.lev_shift = lev_shift; ev.nlg = int(nlg); ev.bins_per_chan = int(bins_per_chan);
            sp.n_tiles = (sp.nbins + kScanTile - 1) / kScanTile;
            CUDA_TRY(g, g->hist.ensure(size_t(sp.nbins) * sizeof(unsigned int)));
            CUDA_TRY(g, g->tile_sums.ensure(size_t(sp.n_tiles) * sizeof(unsigned int)));
            sp.count = ev.count; sp.cap = ev.cap;
            sp.keys = g->evkeys.as<unsigned int>();
            ev.keys = g->evkeys.as<unsigned int>(); ev.hist = emission ? nullptr : g->hist.as<unsigned int>();
            ev.c_fold = sp.c_fold; ev.nlev = g->nlev; ev.nlat = g->nlat; ev.ncell = g->ncell;
            sp.hist = g->hist.as<unsigned int>(); sp.tile_sums = g->tile_sums.as<unsigned int>();
            sp.perm = g->perm.as<unsigned int>();
            sp.nlev = g->nlev; sp.nlat = g->nlat; sp.ncell = g->ncell;
        } else {
            ev.keys = nullptr; ev.hist = nullptr;
        }
        // ---- wavefront kernels (wavefront.cuh): launch geometry and the launch-order sort of albedo runs
        // continuous absorption runs through the persistent kernel only (its march carries the second extinction)
        const int n_gen = cont ? 0 : g->tune[2];
        L.n_gen = n_gen;
        // emission without scattering (L210): the emit kernel has already closed every packet it recorded
        L.n_gen_run = (emission && !prm->scatter_on) ? 0 : n_gen;
        L.k_first = rc.forced_scatter ? wave_first_flight_kernel<16, true> : wave_first_flight_kernel<16, false>;
        L.k_inter = rc.forced_scatter == 2 ? wave_interact_kernel<kInteractK, true> : wave_interact_kernel<kInteractK, false>;
        L.smem_w = smem_t;
        L.smem_i = (size_t((g->tab_floats + 31) & ~31) + size_t(kWaveThreads / 32) * kStageFields * kStageSlots) * sizeof(float);
        L.grid_k = unsigned(g->sm_count * 8);
        SortParams& spl = L.spl;
        if (n_gen > 0) {
            int occ_f = 1, occ_i = 1;
            CUDA_TRY(g, cudaFuncSetAttribute(wave_launch_keys_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, int(L.smem_w)));
            CUDA_TRY(g, cudaFuncSetAttribute(L.k_first, cudaFuncAttributeMaxDynamicSharedMemorySize, int(L.smem_w)));
            CUDA_TRY(g, cudaFuncSetAttribute(wave_emit_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, int(L.smem_w)));
            CUDA_TRY(g, cudaFuncSetAttribute(L.k_inter, cudaFuncAttributeMaxDynamicSharedMemorySize, int(L.smem_i)));
            CUDA_TRY(g, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ_f, L.k_first, kWaveThreads, L.smem_w));
            CUDA_TRY(g, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ_i, L.k_inter, kWaveThreads, L.smem_i));
            if (occ_f < 1 || occ_i < 1) return fail(g, GCMCRT_E_INVALID, "grid tables do not fit in shared memory");
            L.grid_f = unsigned(g->sm_count * occ_f);
            L.grid_i = unsigned(g->sm_count * occ_i);
            CUDA_TRY(g, g->flights.ensure(size_t(g->sm_count) * occ_i * (kWaveThreads / 32) * kFlightFields * kStageSlots * sizeof(float)));
            L.wc.flights = g->flights.as<float>();
            L.wc.c_fold = 1;
            if (!emission) {
                const int ncol = g->nlat * g->nlon;
                // same bound as the event sort: channels a pass can span, and at most 2^25 bins (a run of many channels
                // with few packets each folds the channels beyond the cap into the last slot, which only costs coherence)
                const long long max_lbins = 1ll << 25;
                const long long per_chan = (long long)ncol * kLaunchTauBuckets;
                if (per_chan > max_lbins) return fail(g, GCMCRT_E_INVALID, "grid has too many columns for the launch-order sort");
                spl.c_fold = int(std::max<long long>(1, std::min<long long>(std::min<long long>(ncr, max_lbins / per_chan),
                                                                          (long long)(g->ev_cap / std::max<size_t>(n_pkt, 1)) + 2)));
                spl.nbins = (unsigned int)((long long)spl.c_fold * per_chan);
                spl.n_tiles = (spl.nbins + kScanTile - 1) / kScanTile;
                CUDA_TRY(g, g->lkeys.ensure(size_t(g->ev_cap) * sizeof(unsigned int)));
                CUDA_TRY(g, g->lperm.ensure(size_t(g->ev_cap) * sizeof(unsigned int)));
                CUDA_TRY(g, g->lhist.ensure(size_t(spl.nbins) * sizeof(unsigned int)));
                CUDA_TRY(g, g->ltile.ensure(size_t(spl.n_tiles) * sizeof(unsigned int)));
                spl.keys = g->lkeys.as<unsigned int>(); spl.count = &ctrl->n_fresh; spl.cap = g->ev_cap;
                spl.hist = g->lhist.as<unsigned int>(); spl.tile_sums = g->ltile.as<unsigned int>();
                spl.perm = g->lperm.as<unsigned int>();
                L.wc.keys = g->lkeys.as<unsigned int>(); L.wc.perm = g->lperm.as<unsigned int>();
                L.wc.lhist = spl.hist;   // the launch sort's histogram is counted while the keys are written
                L.wc.c_fold = std::max(spl.c_fold, 1);
            }
        }
        L.tail_items = n_gen > 0 ? 0ull : total_items;   // wavefront: the persistent kernel only finishes what the generations leave over
        L.plan.total_items = total_items; L.plan.susp_cap = susp_cap; L.plan.max_passes = 1ull << 20;
        L.plan.batch0 = std::max<unsigned long long>(1024, g->ev_cap / (unsigned long long)g->tune[3]);
        // emission without scattering: exactly one event per packet, nothing to learn -- the first pass is a full one
        if (emission && !prm->scatter_on) L.plan.batch0 = std::max<unsigned long long>(1024, (unsigned long long)(0.85 * double(g->ev_cap)));
        L.plan.n_pkt = uint32_t(n_pkt); L.plan.ev_cap = g->ev_cap; L.plan.n_gen = n_gen; L.plan.n_chan_run = ncr;
        run_begin_kernel<<<1, 1, 0, s>>>(ctrl, L.plan);
        ++g->launches;
        if (!timed && !host_loop_env) {
            if ((rcode = launch_pass_loop(g, L, s, &launches_per_pass))) return rcode;
        } else {
            for (;;) {
                if ((rcode = enqueue_pass(g, L, s, timed ? g->tev : nullptr, cudaGraphConditionalHandle{}, 0, &launches_per_pass))) return rcode;
                CUDA_TRY(g, cudaMemcpyAsync(g->h_ctrl, ctrl, sizeof(PassCtrl), cudaMemcpyDeviceToHost, s));
                CUDA_TRY(g, cudaStreamSynchronize(s));
                if (timed) {
                    float a = 0.f, b = 0.f, c = 0.f;
                    CUDA_TRY(g, cudaEventElapsedTime(&a, g->tev[0], g->tev[1]));
                    CUDA_TRY(g, cudaEventElapsedTime(&b, g->tev[1], g->tev[2]));
                    CUDA_TRY(g, cudaEventElapsedTime(&c, g->tev[2], g->tev[3]));
                    g->ms_transport += a; g->ms_sort += b; g->ms_peel += c;
                }
                if (g->h_ctrl->error == 1) return fail(g, GCMCRT_E_CUDA, "suspended-packet list overflow");
                if (g->h_ctrl->error) return fail(g, GCMCRT_E_CUDA, "pass loop did not terminate");
                if (g->h_ctrl->done) break;
            }
        }
    }

    // ---- A10
    if (n_obs > 0) {
        const int nt = ncr * n_obs;
        normalise_kernel<<<(nt + 127) / 128, 128, 0, s>>>(ncr, n_obs, nb, N, lo, hi, static_cast<double*>(o_flux.dev),
                                                         static_cast<double*>(o_ltot.dev), mode,
                                                         g->r[g->nlev] - g->r[0],
                                                         static_cast<double*>(o_val.dev), static_cast<double*>(o_sig.dev));
        CUDA_TRY(g, cudaGetLastError());
        ++g->launches;
    }
    g->ms_stage += g->ms_stage_pending;
    g->ms_stage_pending = 0.0;
    if (o_cnt.dev) {
        finalize_counters_kernel<<<1, 1, 0, s>>>(g->counters.as<DevCounters>(), (mode == 2 && !ms_trans) ? nullptr : ctrl,
                                                static_cast<gcmcrt_counters*>(o_cnt.dev), g->launches + 1, launches_per_pass,
                                                passes_host, g->ms_stage, g->ms_emis, g->ms_transport, g->ms_peel, g->ms_sort);
        CUDA_TRY(g, cudaGetLastError());
    }
    // ---- copy-backs for host-resident outputs (the only place an untimed run waits for the device)
    bool need_sync = false;
    for (OutBuf* ob : {&o_flux, &o_ltot, &o_val, &o_sig, &o_img, &o_evc, &o_ctb, &o_cnt}) {
        if (ob->host && ob->dev && ob->bytes) {
            CUDA_TRY(g, cudaMemcpyAsync(ob->host, ob->dev, ob->bytes, cudaMemcpyDeviceToHost, s));
            need_sync = true;
        }
    }
    if (need_sync) {
        CUDA_TRY(g, cudaStreamSynchronize(s));
        reap_retired_loops(g);
    }
    if (o_cnt.host) {
        const unsigned long long st = static_cast<const gcmcrt_counters*>(o_cnt.host)->device_status;
        if (st == 1) return fail(g, GCMCRT_E_CUDA, "suspended-packet list overflow");
        if (st) return fail(g, GCMCRT_E_CUDA, "pass loop did not terminate");
    }
    return GCMCRT_OK;
}

__global__ void sum_counters_kernel(const gcmcrt_counters* part, int k, gcmcrt_counters* out)
{
    gcmcrt_counters a = part[0];
    for (int q = 1; q < k; ++q) {
        const gcmcrt_counters b = part[q];
        a.events += b.events; a.segments_transport += b.segments_transport; a.segments_peel += b.segments_peel;
        a.packets_escaped += b.packets_escaped; a.packets_absorbed += b.packets_absorbed; a.packets_surface += b.packets_surface;
        a.packets_stuck += b.packets_stuck; a.escaped_weight += b.escaped_weight; a.passes += b.passes; a.rays_peel += b.rays_peel;
        a.launches += b.launches; a.ms_stage += b.ms_stage; a.ms_emission_cdf += b.ms_emission_cdf;
        a.ms_transport += b.ms_transport; a.ms_peel += b.ms_peel; a.ms_sort += b.ms_sort;
        a.device_status = a.device_status ? a.device_status : b.device_status;
    }
    *out = a;
}

// run_params.concurrency = K > 1 (L79: the channels of a run are independent): the run's channels are cut into K
// contiguous parts; part 0 runs on this handle and the caller's stream, the others on internal handles -- copies of the
// grid with working buffers of their own, which borrow this handle's opacity tables -- and internal streams that fork
// from the caller's stream and join it again.  Every part is an ordinary run_mode() call with device outputs that point
// into the whole run's arrays, so the parts are only enqueued; what the caller wants in host memory is copied back after
// the join.  The kernels of one part fill the issue slots and the memory latencies another leaves idle.
bool split_eligible(gcmcrt_grid* g, const gcmcrt_run_params* prm, const gcmcrt_result* out, cudaStream_t s, int mode)
{
    if (!g || !prm || !out || g->is_peer || prm->concurrency < 2 || prm->concurrency > 8) return false;
    if (mode == 2 || prm->timing || g->n_chan <= 0 || g->staged_obs == -2) return false;
    static const bool host_loop_env = std::getenv("GCMCRT_HOST_LOOP") && std::atoi(std::getenv("GCMCRT_HOST_LOOP")) != 0;
    if (host_loop_env) return false;
    const int cb = prm->chan_begin, ce = prm->chan_end ? prm->chan_end : g->n_chan;
    if (cb < 0 || ce > g->n_chan || ce - cb < prm->concurrency) return false;
    const unsigned long long N = prm->packets_per_channel, lo = prm->pkt_begin, hi = prm->pkt_end ? prm->pkt_end : N;
    if (N == 0 || N > 0xffffffffull || lo > hi || hi > N) return false;       // run_mode() reports it
    if (prm->n_obs < 0 || prm->n_obs > kMaxObs || (prm->n_obs > 0 && !out->flux_sum)) return false;
    const int nb = prm->n_batches ? prm->n_batches : 32;
    if (nb < 1 || nb > kMaxBatches) return false;
    cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
    if (cudaStreamIsCapturing(s, &cs) != cudaSuccess) { cudaGetLastError(); return false; }
    return cs == cudaStreamCaptureStatusNone;
}

int run_split(gcmcrt_grid* g, const gcmcrt_run_params* prm, gcmcrt_result* out, void* stream, int mode)
{
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    const int K = prm->concurrency;
    const int n_obs = prm->n_obs, nobs1 = std::max(n_obs, 1);
    const unsigned long long N = prm->packets_per_channel, lo = prm->pkt_begin, hi = prm->pkt_end ? prm->pkt_end : N;
    const int cb = prm->chan_begin, ce = prm->chan_end ? prm->chan_end : g->n_chan, ncr = ce - cb;
    const int nb = prm->n_batches ? prm->n_batches : 32;
    const int npix = prm->npix > 0 && out->image ? prm->npix : 0;
    const size_t n_pkt = size_t(hi - lo);
    int rcode;
    // ---- internal handles and their streams (created once: the first call of this kind waits for the device)
    while (int(g->peers.size()) < K - 1) {
        gcmcrt_grid* p = nullptr;
        rcode = gcmcrt_grid_create(&p, g->nlev, g->nlat, g->nlon, g->r.data(), g->th.data(), g->ph.data(), g->T.as<float>(),
                                   g->rho.as<float>(), g->u.p ? g->u.as<float>() : nullptr, g->v.p ? g->v.as<float>() : nullptr,
                                   g->w.p ? g->w.as<float>() : nullptr, g->Omega, g->surface_albedo, s);
        if (rcode) return fail(g, rcode, "concurrency: " + g_create_error);
        p->is_peer = true;
        p->owner = g;
        cudaStream_t ps = nullptr;
        cudaEvent_t pe = nullptr;
        cudaError_t e = cudaStreamCreateWithFlags(&ps, cudaStreamNonBlocking);
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&pe, cudaEventDisableTiming);
        if (e != cudaSuccess) { gcmcrt_destroy(p); if (ps) cudaStreamDestroy(ps); cudaGetLastError(); return fail(g, GCMCRT_E_CUDA, "concurrency: stream"); }
        g->peers.push_back(p); g->peer_streams.push_back(ps); g->peer_done.push_back(pe);
    }
    if (!g->fork_ev) CUDA_TRY(g, cudaEventCreateWithFlags(&g->fork_ev, cudaEventDisableTiming));
    CUDA_TRY(g, g->part_counters.ensure(size_t(K) * sizeof(gcmcrt_counters)));
    // ---- outputs of the whole run, bound once (host-resident ones are staged on this handle)
    OutBuf o_flux, o_ltot, o_val, o_sig, o_img, o_evc, o_ctb, o_cnt;
    if ((rcode = bind_out(g, out->flux_sum, size_t(ncr) * nobs1 * nb * sizeof(double), g->flux, o_flux))) return rcode;
    if ((rcode = bind_out(g, out->L_tot, size_t(ncr) * nobs1 * sizeof(double), g->ltot_out, o_ltot))) return rcode;
    if ((rcode = bind_out(g, out->value, size_t(ncr) * nobs1 * sizeof(double), g->value, o_val))) return rcode;
    if ((rcode = bind_out(g, out->sigma, size_t(ncr) * nobs1 * sizeof(double), g->sigma, o_sig))) return rcode;
    if (npix) if ((rcode = bind_out(g, out->image, size_t(ncr) * n_obs * npix * npix * sizeof(float), g->image, o_img))) return rcode;
    if (out->event_count) if ((rcode = bind_out(g, out->event_count, size_t(ncr) * n_pkt * sizeof(uint32_t), g->evcount, o_evc))) return rcode;
    if (out->contrib && n_obs > 0) if ((rcode = bind_out(g, out->contrib, size_t(ncr) * n_obs * 2 * g->ncell * sizeof(float), g->contrib, o_ctb))) return rcode;
    if (out->counters) if ((rcode = bind_out(g, out->counters, sizeof(gcmcrt_counters), g->counters_out, o_cnt))) return rcode;
    // ---- fork: the internal streams wait for everything enqueued on the caller's stream (its table copies included)
    CUDA_TRY(g, cudaEventRecord(g->fork_ev, s));
    for (int q = 1; q < K; ++q) CUDA_TRY(g, cudaStreamWaitEvent(g->peer_streams[q - 1], g->fork_ev, 0));
    for (int q = 1; q < K; ++q) {
        gcmcrt_grid* p = g->peers[q - 1];
        if (p->synced_epoch == g->opacity_epoch) continue;
        rcode = g->use_nodes
                    ? gcmcrt_set_opacity_nodes(p, g->chan0, g->n_chan, g->lambda.data(), g->node.as<float>(), g->nT, g->nP, g->T_nodes_h.data(),
                                               g->logp_nodes_h.data(), g->own_pcell.as<float>(), g->k_ray, g->k_cld, g->g_cld, g->peer_streams[q - 1])
                    : gcmcrt_set_opacity(p, g->chan0, g->n_chan, g->lambda.data(), g->k_abs, g->k_ray, g->k_cld, g->g_cld, g->peer_streams[q - 1]);
        if (rcode) return fail(g, rcode, "concurrency: " + p->err);
        p->synced_epoch = g->opacity_epoch;   // (of the handle it borrows from)
    }
    // ---- the parts
    int first_err = GCMCRT_OK;
    for (int q = 0; q < K && first_err == GCMCRT_OK; ++q) {
        const int c0 = cb + int((long long)ncr * q / K), c1 = cb + int((long long)ncr * (q + 1) / K);
        const size_t oc = size_t(c0 - cb);
        gcmcrt_run_params pq = *prm;
        pq.chan_begin = c0; pq.chan_end = c1; pq.concurrency = 0;
        gcmcrt_result rq;
        std::memset(&rq, 0, sizeof rq);
        rq.flux_sum = static_cast<double*>(o_flux.dev) + oc * nobs1 * nb;
        rq.L_tot = static_cast<double*>(o_ltot.dev) + oc * nobs1;
        rq.value = static_cast<double*>(o_val.dev) + oc * nobs1;
        rq.sigma = static_cast<double*>(o_sig.dev) + oc * nobs1;
        rq.image = npix ? static_cast<float*>(o_img.dev) + oc * n_obs * npix * npix : nullptr;
        rq.event_count = o_evc.dev ? static_cast<uint32_t*>(o_evc.dev) + oc * n_pkt : nullptr;
        rq.contrib = o_ctb.dev ? static_cast<float*>(o_ctb.dev) + oc * n_obs * 2 * g->ncell : nullptr;
        rq.counters = g->part_counters.as<gcmcrt_counters>() + q;
        gcmcrt_grid* h = q == 0 ? g : g->peers[q - 1];
        rcode = run_mode(h, &pq, &rq, q == 0 ? s : g->peer_streams[q - 1], mode, true);
        if (rcode) { first_err = rcode; if (h != g) g->err = "concurrency: " + h->err; }
    }
    // ---- join (also after a failed part: nothing may be left running behind the caller's back)
    for (int q = 1; q < K; ++q) {
        CUDA_TRY(g, cudaEventRecord(g->peer_done[q - 1], g->peer_streams[q - 1]));
        CUDA_TRY(g, cudaStreamWaitEvent(s, g->peer_done[q - 1], 0));
    }
    if (first_err) return first_err;
    if (o_cnt.dev) {
        sum_counters_kernel<<<1, 1, 0, s>>>(g->part_counters.as<gcmcrt_counters>(), K, static_cast<gcmcrt_counters*>(o_cnt.dev));
        CUDA_TRY(g, cudaGetLastError());
    }
    bool need_sync = false;
    for (OutBuf* ob : {&o_flux, &o_ltot, &o_val, &o_sig, &o_img, &o_evc, &o_ctb, &o_cnt}) {
        if (ob->host && ob->dev && ob->bytes) {
            CUDA_TRY(g, cudaMemcpyAsync(ob->host, ob->dev, ob->bytes, cudaMemcpyDeviceToHost, s));
            need_sync = true;
        }
    }
    if (need_sync) {
        CUDA_TRY(g, cudaStreamSynchronize(s));
        reap_retired_loops(g);
        for (gcmcrt_grid* p : g->peers) reap_retired_loops(p);
    }
    if (o_cnt.host) {
        const unsigned long long st = static_cast<const gcmcrt_counters*>(o_cnt.host)->device_status;
        if (st == 1) return fail(g, GCMCRT_E_CUDA, "suspended-packet list overflow");
        if (st) return fail(g, GCMCRT_E_CUDA, "pass loop did not terminate");
    }
    return GCMCRT_OK;
}

int run_entry(gcmcrt_grid* g, const gcmcrt_run_params* prm, gcmcrt_result* out, void* stream, int mode)
{
    if (split_eligible(g, prm, out, static_cast<cudaStream_t>(stream), mode)) return run_split(g, prm, out, stream, mode);
    return run_mode(g, prm, out, stream, mode);
}

}  // namespace

extern "C" {

const char* gcmcrt_version(void) { return "gcmcrt 0.1 sm_100a (CUDA " "12.9" ")"; }

const char* gcmcrt_last_error(const gcmcrt_grid* grid) { return grid ? grid->err.c_str() : g_create_error.c_str(); }

int gcmcrt_grid_create(gcmcrt_grid** out, int nlev, int nlat, int nlon, const double* r_edges, const double* colat_edges,
                       const double* lon_edges, const float* T, const float* rho, const float* u, const float* v,
                       const float* w, double Omega, float surface_albedo, void* stream)
{
    if (!out) return fail(nullptr, GCMCRT_E_INVALID, "out is NULL");
    *out = nullptr;
    if (nlev < 1 || nlat < 1 || nlon < 1 || nlev > 1023 || nlat > 1023 || nlon > 2047)
        return fail(nullptr, GCMCRT_E_INVALID, "grid sizes must satisfy 1 <= nlev, nlat <= 1023, 1 <= nlon <= 2047");
    if (!r_edges || !colat_edges || !lon_edges || !T || !rho) return fail(nullptr, GCMCRT_E_INVALID, "NULL grid array");
    for (int i = 0; i < nlev; ++i)
        if (!(r_edges[i + 1] > r_edges[i]) || !(r_edges[i] > 0.0)) return fail(nullptr, GCMCRT_E_INVALID, "r_edges must be positive and strictly ascending");
    for (int j = 0; j < nlat; ++j)
        if (!(colat_edges[j + 1] > colat_edges[j])) return fail(nullptr, GCMCRT_E_INVALID, "colat_edges must be strictly ascending");
    for (int k = 0; k < nlon; ++k)
        if (!(lon_edges[k + 1] > lon_edges[k])) return fail(nullptr, GCMCRT_E_INVALID, "lon_edges must be strictly ascending");
    const double pi = 3.14159265358979323846;
    if (std::fabs(colat_edges[0]) > 1e-9 || std::fabs(colat_edges[nlat] - pi) > 1e-9)
        return fail(nullptr, GCMCRT_E_INVALID, "colat_edges must span 0..pi");
    if (std::fabs(lon_edges[0]) > 1e-9 || std::fabs(lon_edges[nlon] - 2 * pi) > 1e-9)
        return fail(nullptr, GCMCRT_E_INVALID, "lon_edges must span 0..2pi");
    if (!(surface_albedo >= 0.f && surface_albedo <= 1.f)) return fail(nullptr, GCMCRT_E_INVALID, "surface_albedo must be in [0,1]");
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) { cudaGetLastError(); return fail(nullptr, GCMCRT_E_CUDA, "no CUDA device"); }
    gcmcrt_grid* g = new (std::nothrow) gcmcrt_grid;
    if (!g) return fail(nullptr, GCMCRT_E_NOMEM, "host allocation failed");
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    g->nlev = nlev; g->nlat = nlat; g->nlon = nlon; g->ncell = nlev * nlat * nlon;
    g->r.assign(r_edges, r_edges + nlev + 1);
    g->th.assign(colat_edges, colat_edges + nlat + 1);
    g->ph.assign(lon_edges, lon_edges + nlon + 1);
    g->Omega = Omega; g->surface_albedo = surface_albedo;
    cudaDeviceGetAttribute(&g->sm_count, cudaDevAttrMultiProcessorCount, dev);

    // packed fp32 tables: R^2 (high, low) pairs, R, qcube, cos(theta_e), cos(phi_e), sin(phi_e), phi_e
    std::vector<float> tab;
    for (int i = 0; i <= nlev; ++i) {   // R_k^2 as (high, low) pairs: one LDS.64 per shell root
        const double r2 = g->r[i] * g->r[i];
        tab.push_back(float(r2));
        tab.push_back(float(r2 - double(float(r2))));
    }
    for (int i = 0; i <= nlev; ++i) tab.push_back(float(g->r[i]));
    for (int i = 0; i < nlev; ++i) { const double q = g->r[i + 1] / g->r[i]; tab.push_back(float(q * q * q - 1.0)); }
    std::vector<double> cth(nlat + 1);
    for (int j = 0; j <= nlat; ++j) cth[j] = j == 0 ? 1.0 : (j == nlat ? -1.0 : std::cos(g->th[j]));
    for (int j = 0; j <= nlat; ++j) tab.push_back(float(cth[j]));
    for (int k = 0; k <= nlon; ++k) tab.push_back(float(k == nlon ? std::cos(g->ph[0]) : std::cos(g->ph[k])));
    for (int k = 0; k <= nlon; ++k) tab.push_back(float(k == nlon ? std::sin(g->ph[0]) : std::sin(g->ph[k])));
    for (int k = 0; k <= nlon; ++k) tab.push_back(float(g->ph[k]));
    g->tab_floats = int(tab.size());
    std::vector<float> rc(nlev), thc(nlat), phc(nlon);
    for (int i = 0; i < nlev; ++i) rc[i] = float(0.5 * (g->r[i] + g->r[i + 1]));
    for (int j = 0; j < nlat; ++j) thc[j] = float(0.5 * (g->th[j] + g->th[j + 1]));
    for (int k = 0; k < nlon; ++k) phc[k] = float(0.5 * (g->ph[k] + g->ph[k + 1]));

    cudaError_t e = upload(g->tab, tab, s);
    if (e == cudaSuccess) e = upload(g->r64, g->r, s);
    if (e == cudaSuccess) e = upload(g->cth64, cth, s);
    if (e == cudaSuccess) e = upload(g->ph64, g->ph, s);
    if (e == cudaSuccess) e = upload(g->rc32, rc, s);
    if (e == cudaSuccess) e = upload(g->thc32, thc, s);
    if (e == cudaSuccess) e = upload(g->phc32, phc, s);
    const float* dummy = nullptr;
    const size_t nc = size_t(g->ncell);
    if (e == cudaSuccess) e = device_view(T, nc, g->T, s, &dummy, true);
    if (e == cudaSuccess) e = device_view(rho, nc, g->rho, s, &dummy, true);
    if (e == cudaSuccess && u) e = device_view(u, nc, g->u, s, &dummy, true);
    if (e == cudaSuccess && v) e = device_view(v, nc, g->v, s, &dummy, true);
    if (e == cudaSuccess && w) e = device_view(w, nc, g->w, s, &dummy, true);
    if (e == cudaSuccess) e = cudaStreamSynchronize(s);   // host vectors above go out of scope
    if (e != cudaSuccess) {
        const int code = fail(nullptr, e == cudaErrorMemoryAllocation ? GCMCRT_E_NOMEM : GCMCRT_E_CUDA,
                              std::string("grid_create: ") + cudaGetErrorString(e));
        cudaGetLastError();
        gcmcrt_destroy(g);
        return code;
    }
    *out = g;
    return GCMCRT_OK;
}

static int set_opacity_common(gcmcrt_grid* g, int chan0, int n_chan, const float* lambda, const float* k_sca_ray,
                              const float* k_sca_cld, const float* g_cld, cudaStream_t s);

int gcmcrt_set_opacity(gcmcrt_grid* g, int chan0, int n_chan, const float* lambda, const float* k_abs,
                       const float* k_sca_ray, const float* k_sca_cld, const float* g_cld, void* stream)
{
    if (!g) return GCMCRT_E_INVALID;
    if (n_chan < 1 || chan0 < 0 || !lambda || !k_abs) return fail(g, GCMCRT_E_INVALID, "set_opacity: bad arguments");
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    const size_t n = size_t(n_chan) * g->ncell;
    g->staged_obs = -2;
    g->n_chan = 0;
    g->use_nodes = false;
    CUDA_TRY(g, device_view(k_abs, n, g->own_kabs, s, &g->k_abs));
    return set_opacity_common(g, chan0, n_chan, lambda, k_sca_ray, k_sca_cld, g_cld, s);
}

int gcmcrt_set_opacity_nodes(gcmcrt_grid* g, int chan0, int n_chan, const float* lambda, const float* node_kabs, int nT,
                             int nP, const float* T_nodes, const float* logp_nodes, const float* p_cell,
                             const float* k_sca_ray, const float* k_sca_cld, const float* g_cld, void* stream)
{
    if (!g) return GCMCRT_E_INVALID;
    if (n_chan < 1 || chan0 < 0 || !lambda || !node_kabs || nT < 2 || nP < 2 || !T_nodes || !logp_nodes || !p_cell)
        return fail(g, GCMCRT_E_INVALID, "set_opacity_nodes: bad arguments");
    const float dT = (T_nodes[nT - 1] - T_nodes[0]) / float(nT - 1), dlp = (logp_nodes[nP - 1] - logp_nodes[0]) / float(nP - 1);
    if (!(dT > 0.f) || !(dlp > 0.f)) return fail(g, GCMCRT_E_INVALID, "set_opacity_nodes: node axes must ascend");
    for (int a = 1; a < nT; ++a)
        if (std::fabs((T_nodes[a] - T_nodes[a - 1]) - dT) > 1e-3f * dT) return fail(g, GCMCRT_E_INVALID, "set_opacity_nodes: T_nodes must be uniformly spaced");
    for (int b = 1; b < nP; ++b)
        if (std::fabs((logp_nodes[b] - logp_nodes[b - 1]) - dlp) > 1e-3f * dlp) return fail(g, GCMCRT_E_INVALID, "set_opacity_nodes: logp_nodes must be uniformly spaced");
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    g->staged_obs = -2;
    g->n_chan = 0;
    g->k_abs = nullptr;
    const float* dnode = nullptr;
    const float* dp = nullptr;
    CUDA_TRY(g, device_view(node_kabs, size_t(n_chan) * nT * nP, g->node, s, &dnode, true));
    CUDA_TRY(g, device_view(p_cell, size_t(g->ncell), g->own_pcell, s, &dp, true));
    CUDA_TRY(g, g->node_idx.ensure(size_t(g->ncell) * sizeof(int2)));
    CUDA_TRY(g, g->node_w.ensure(size_t(g->ncell) * sizeof(float2)));
    node_coeff_kernel<<<(g->ncell + 255) / 256, 256, 0, s>>>(g->ncell, g->T.as<float>(), dp, T_nodes[0], dT, logp_nodes[0], dlp,
                                                            nT, nP, g->node_idx.as<int2>(), g->node_w.as<float2>());
    CUDA_TRY(g, cudaGetLastError());
    g->nT = nT; g->nP = nP;
    g->T_nodes_h.assign(T_nodes, T_nodes + nT); g->logp_nodes_h.assign(logp_nodes, logp_nodes + nP);   // for the internal handles
    g->use_nodes = true;
    return set_opacity_common(g, chan0, n_chan, lambda, k_sca_ray, k_sca_cld, g_cld, s);
}

static int set_opacity_common(gcmcrt_grid* g, int chan0, int n_chan, const float* lambda, const float* k_sca_ray,
                              const float* k_sca_cld, const float* g_cld, cudaStream_t s)
{
    const size_t n = size_t(n_chan) * g->ncell;
    CUDA_TRY(g, device_view(k_sca_ray, n, g->own_kray, s, &g->k_ray));
    CUDA_TRY(g, device_view(k_sca_cld, n, g->own_kcld, s, &g->k_cld));
    CUDA_TRY(g, device_view(g_cld, n, g->own_g, s, &g->g_cld));
    std::vector<float> lam(n_chan);
    if (is_device_ptr(lambda)) {
        CUDA_TRY(g, cudaMemcpyAsync(lam.data(), lambda, n_chan * sizeof(float), cudaMemcpyDeviceToHost, s));
        CUDA_TRY(g, cudaStreamSynchronize(s));
    } else {
        std::memcpy(lam.data(), lambda, n_chan * sizeof(float));
    }
    for (int c = 0; c < n_chan; ++c)
        if (!(lam[c] > 0.f)) return fail(g, GCMCRT_E_INVALID, "lambda must be positive");
    g->lambda = lam;
    // staging vectors owned by the handle: the uploads below are asynchronous
    std::vector<double>& lam64 = g->lambda64_h;
    std::vector<float>& reff = g->reff_h;
    lam64.assign(lam.begin(), lam.end());
    reff.assign(n_chan, 0.f);
    for (int c = 0; c < n_chan && n_chan > 1; ++c) {
        const int c1 = c + 1 < n_chan ? c : c - 1;
        const double ratio = double(lam[c1 + 1]) / double(lam[c1]);
        reff[c] = ratio != 1.0 ? float(1.0 / std::log(ratio)) : 0.f;
    }
    if (g->owner && g->owner->lambda64.p && g->owner->reff.p && g->owner->n_chan == n_chan) {
        // an internal handle takes the two per-channel arrays from its owner on the device: an upload from pageable host
        // memory of more than 64 KB waits for the stream, which is still running the previous run's part
        CUDA_TRY(g, g->lambda64.ensure(size_t(n_chan) * sizeof(double)));
        CUDA_TRY(g, g->reff.ensure(size_t(n_chan) * sizeof(float)));
        CUDA_TRY(g, cudaMemcpyAsync(g->lambda64.p, g->owner->lambda64.p, size_t(n_chan) * sizeof(double), cudaMemcpyDeviceToDevice, s));
        CUDA_TRY(g, cudaMemcpyAsync(g->reff.p, g->owner->reff.p, size_t(n_chan) * sizeof(float), cudaMemcpyDeviceToDevice, s));
    } else {
        CUDA_TRY(g, upload(g->lambda64, lam64, s));
        CUDA_TRY(g, upload(g->reff, reff, s));
    }
    g->chan0 = chan0;
    g->n_chan = n_chan;
    ++g->opacity_epoch;
    g->launches = 0;
    g->ms_stage_pending = 0.0;
    // staging (A0 / A1) is left to the first run: a Doppler run needs the table of its own observer, not the unshifted one
    g->staged_obs = -3;
    g->launches_pending = 0;
    return GCMCRT_OK;
}

int gcmcrt_run_albedo(gcmcrt_grid* g, const gcmcrt_run_params* p, gcmcrt_result* out, void* stream)
{
    return run_entry(g, p, out, stream, 0);
}

int gcmcrt_run_emission(gcmcrt_grid* g, const gcmcrt_run_params* p, gcmcrt_result* out, void* stream)
{
    return run_entry(g, p, out, stream, 1);
}

int gcmcrt_run_transmission(gcmcrt_grid* g, const gcmcrt_run_params* p, gcmcrt_result* out, void* stream)
{
    return run_entry(g, p, out, stream, 2);
}

int gcmcrt_destroy(gcmcrt_grid* g)
{
    if (!g) return GCMCRT_OK;
    cudaDeviceSynchronize();
    cudaGetLastError();
    for (DevBuf* b : {&g->tab, &g->r64, &g->cth64, &g->ph64, &g->rc32, &g->thc32, &g->phc32, &g->T, &g->rho, &g->u, &g->v,
                      &g->w, &g->own_kabs, &g->own_kray, &g->own_kcld, &g->own_g, &g->alpha, &g->alpha2, &g->prop, &g->reff, &g->vlos, &g->node, &g->node_idx, &g->node_w, &g->own_pcell,
                      &g->lambda64, &g->Lcell, &g->Lcum, &g->Lcol, &g->Ltot, &g->guide, &g->ev0, &g->evkeys, &g->perm, &g->hist, &g->tile_sums, &g->lkeys, &g->lperm, &g->lhist, &g->ltile, &g->flights, &g->s0[0], &g->s0[1],
                      &g->s1[0], &g->s1[1], &g->s2[0], &g->s2[1], &g->ctrl, &g->counters, &g->counters_out, &g->flux, &g->ltot_out,
                      &g->value, &g->sigma, &g->image, &g->evcount, &g->contrib})
        b->release();
    for (gcmcrt_grid* p : g->peers) gcmcrt_destroy(p);
    g->peers.clear();
    for (cudaStream_t ps : g->peer_streams) cudaStreamDestroy(ps);
    for (cudaEvent_t pe : g->peer_done) cudaEventDestroy(pe);
    if (g->fork_ev) cudaEventDestroy(g->fork_ev);
    g->part_counters.release();
    if (g->h_ctrl) cudaFreeHost(g->h_ctrl);
    for (auto& lg : g->loops) g->retired.push_back(lg);
    g->loops.clear();
    reap_retired_loops(g);
    if (g->cap_stream) cudaStreamDestroy(g->cap_stream);
    for (auto& e : g->tev) if (e) cudaEventDestroy(e);
    delete g;
    return GCMCRT_OK;
}

int gcmcrt_debug_ray_tau(gcmcrt_grid* g, int chan, long n, const float* pos, const float* dir, float* tau,
                         int* hit_surface, void* stream)
{
    if (!g) return GCMCRT_E_INVALID;
    if (g->staged_obs == -2) return fail(g, GCMCRT_E_STATE, "gcmcrt_set_opacity has not been called");
    if (chan < 0 || chan >= g->n_chan || n < 0 || !pos || !dir || !tau) return fail(g, GCMCRT_E_INVALID, "debug_ray_tau: bad arguments");
    if (n == 0) return GCMCRT_OK;
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    if (g->staged_obs == -3) { const int rs = stage_opacity(g, nullptr, 0, s); if (rs) return rs; }
    DevBuf bp, bd, bt, bh;
    const float *dp = nullptr, *dd = nullptr;
    int rcode = GCMCRT_OK;
    do {
        cudaError_t e = device_view(pos, size_t(3 * n), bp, s, &dp);
        if (e == cudaSuccess) e = device_view(dir, size_t(3 * n), bd, s, &dd);
        const bool tdev = is_device_ptr(tau), hdev = hit_surface && is_device_ptr(hit_surface);
        float* dt = tau; int* dh = hit_surface;
        if (e == cudaSuccess && !tdev) { e = bt.ensure(n * sizeof(float)); dt = bt.as<float>(); }
        if (e == cudaSuccess && hit_surface && !hdev) { e = bh.ensure(n * sizeof(int)); dh = bh.as<int>(); }
        if (e == cudaSuccess) {
            const GeomParams gp = geom_params(g);
            debug_ray_tau_kernel<<<(unsigned)((n + 127) / 128), 128, g->tab_floats * sizeof(float), s>>>(
                gp, g->alpha.as<float>() + size_t(chan) * size_t(gp.alpha_stride), n, dp, dd, dt, dh);
            e = cudaGetLastError();
        }
        if (e == cudaSuccess && !tdev) e = cudaMemcpyAsync(tau, dt, n * sizeof(float), cudaMemcpyDeviceToHost, s);
        if (e == cudaSuccess && hit_surface && !hdev) e = cudaMemcpyAsync(hit_surface, dh, n * sizeof(int), cudaMemcpyDeviceToHost, s);
        if (e == cudaSuccess) e = cudaStreamSynchronize(s);
        if (e != cudaSuccess) rcode = fail(g, GCMCRT_E_CUDA, std::string("debug_ray_tau: ") + cudaGetErrorString(e));
    } while (0);
    bp.release(); bd.release(); bt.release(); bh.release();
    return rcode;
}

int gcmcrt_debug_philox(long n, const uint32_t* ctr, const uint32_t* key, uint32_t* out, void* stream)
{
    if (n < 0 || !ctr || !key || !out) return GCMCRT_E_INVALID;
    if (n == 0) return GCMCRT_OK;
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    DevBuf bc, bk, bo;
    const uint32_t *dc = nullptr, *dk = nullptr;
    cudaError_t e = device_view(ctr, size_t(4 * n), bc, s, &dc);
    if (e == cudaSuccess) e = device_view(key, size_t(2 * n), bk, s, &dk);
    const bool odev = is_device_ptr(out);
    uint32_t* dout = out;
    if (e == cudaSuccess && !odev) { e = bo.ensure(size_t(4 * n) * sizeof(uint32_t)); dout = bo.as<uint32_t>(); }
    if (e == cudaSuccess) {
        debug_philox_kernel<<<(unsigned)((n + 127) / 128), 128, 0, s>>>(n, dc, dk, dout);
        e = cudaGetLastError();
    }
    if (e == cudaSuccess && !odev) e = cudaMemcpyAsync(out, dout, size_t(4 * n) * sizeof(uint32_t), cudaMemcpyDeviceToHost, s);
    if (e == cudaSuccess) e = cudaStreamSynchronize(s);
    bc.release(); bk.release(); bo.release();
    if (e != cudaSuccess) { g_create_error = std::string("debug_philox: ") + cudaGetErrorString(e); cudaGetLastError(); return GCMCRT_E_CUDA; }
    return GCMCRT_OK;
}

// ---------------------------------------------------------------------------------------------------------
// gcmcrt_emission_ltot_static: total luminosities (Eq. 27 summed over the cells, depth cut of L210) of the staged
// tables with NO allocation -- for callers that must not reach cudaMalloc (code under stream capture, serving loops,
// harnesses that forbid it).  The per-column totals, which gcmcrt_run_emission keeps in a buffer of the handle that
// grows on demand, live in a file-scope device array of fixed size here.  Every GPU that loads the library holds
// the array until the process exits; every call shares it, so calls that overlap on the GPU race.
// ---------------------------------------------------------------------------------------------------------
}  // extern "C"

namespace {

constexpr size_t kStaticScratchBytes = size_t(GCMCRT_STATIC_SCRATCH_BYTES);
static __device__ __align__(256) unsigned char g_static_scratch[kStaticScratchBytes];

// Device address of g_static_scratch on the current device.  In host code the array's name is only a handle for the
// runtime, not a device address: cudaGetSymbolAddress translates it, once per device, with that device current.
cudaError_t static_scratch_address(void** out)
{
    constexpr int kMaxDevices = 64;
    static void* ptr[kMaxDevices] = {};
    static std::mutex mtx;
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= kMaxDevices) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(mtx);
    if (!ptr[dev]) {
        void* p = nullptr;
        e = cudaGetSymbolAddress(&p, g_static_scratch);
        if (e != cudaSuccess) return e;
        ptr[dev] = p;
    }
    *out = ptr[dev];
    return cudaSuccess;
}

// emis_col_kernel without its table outputs: the same loads, depth cut, L_i (Eq. 27) and fp64 warp scan in the same
// order -- so the column totals are bit-identical -- and one store per (channel, column): the column's total into
// col_tot[c_rel][col] (the static scratch).  p.alpha, p.prop, p.lambda point at the first channel of the range,
// p.n_chan is the number of channels.
template <int NCH>
__global__ void __launch_bounds__(kEmisThreads) emis_coltot_static_kernel(const EmisParams p, double* __restrict__ col_tot)
{
    extern __shared__ double emis_sm[];
    double* dr = emis_sm;
    double* dr3 = dr + p.nlev;
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
        const double hck = 6.62607015e-34 * 299792458.0 / (lam * 1.380649e-23);
        const double pre = 4.0 * 3.14159265358979323846 * 2.0 * 6.62607015e-34 * 299792458.0 * 299792458.0 /
                           (lam * lam * lam * lam * lam);
        const float* alpha_c = p.alpha + (size_t)c * p.alpha_stride;
        const float4* prop_c = p.prop + (size_t)c * p.ncell;
        for (int col = blockIdx.x * (kEmisThreads / 32) + wid; col < ncol; col += gridDim.x * (kEmisThreads / 32)) {
            const size_t cell0 = (size_t)col * p.nlev;
            const float* acol = alpha_c + (size_t)col * p.col_stride + 1;
            float a[NCH], T[NCH];
            double rk[NCH];   // rho kappa_abs: the fp64 product of two fp32 values is exact, as in the oracle's fp64
#pragma unroll
            for (int m = 0; m < NCH; ++m) {
                const int i = (m << 5) + lane;
                const bool in = i < p.nlev;
                a[m] = in ? __ldg(acol + i) : 0.0f;
                T[m] = in ? __ldg(p.T + cell0 + i) : 1.0f;
                rk[m] = in ? double(__ldg(p.rho + cell0 + i)) * double(__ldg(&prop_c[cell0 + i].w)) : 0.0;
            }
            int i_cut = 0;
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
                    if (mc) i_cut = (m << 5) + 32 - __clz(mc);
                }
            }
            const int j = col % p.nlat, k = col / p.nlat;
            const double ang = (p.cth_edges[j] - p.cth_edges[j + 1]) * (p.ph_edges[k + 1] - p.ph_edges[k]);
            double run = 0.0;
#pragma unroll
            for (int m = 0; m < NCH; ++m) {
                const int i = (m << 5) + lane;
                if ((m << 5) + 32 > i_cut && (m << 5) < p.nlev) {
                    double Li = 0.0;
                    if (i < p.nlev && i >= i_cut) {
                        const double e = expm1(hck * rcp_pos_f64(double(T[m])));
                        Li = e < 1e300 ? pre * dr3[i] * ang * rk[m] * rcp_pos_f64(e) : 0.0;
                    }
                    const double sum = run + warp_incl_scan_f64(Li);
                    run = __shfl_sync(kFullMask, sum, 31);
                }
            }
            if (lane == 0) col_tot[(size_t)c * ncol + col] = run;
        }
    }
}

}  // namespace

extern "C" {

int gcmcrt_emission_ltot_static(gcmcrt_grid* g, int chan_begin, int chan_end, double tau_vert_max, double* L_tot, void* stream)
{
    if (!g) return GCMCRT_E_INVALID;
    if (!L_tot) return fail(g, GCMCRT_E_INVALID, "emission_ltot_static: L_tot is NULL");
    if (g->n_chan <= 0 || g->staged_obs < -1)
        return fail(g, GCMCRT_E_STATE, "emission_ltot_static: no staged tables (they are staged by the first run after gcmcrt_set_opacity*; "
                                       "this call allocates nothing and therefore stages nothing)");
    const int cb = chan_begin, ce = chan_end ? chan_end : g->n_chan;
    if (cb < 0 || ce > g->n_chan || cb >= ce) return fail(g, GCMCRT_E_INVALID, "emission_ltot_static: bad channel range");
    if (cb < g->staged_c0 || ce > g->staged_c1) return fail(g, GCMCRT_E_STATE, "emission_ltot_static: the staged tables do not hold these channels");
    if (g->nlev > 256) return fail(g, GCMCRT_E_INVALID, "emission: nlev > 256 is not supported");
    const int ncr = ce - cb, ncol = g->nlat * g->nlon;
    // scratch: column totals [ncr][ncol], then the totals [ncr] (copied out when L_tot is host memory)
    const size_t need = (size_t(ncr) * ncol + size_t(ncr)) * sizeof(double);
    if (need > kStaticScratchBytes) {
        char msg[256];
        std::snprintf(msg, sizeof msg, "emission_ltot_static: %d channels x %d columns need %zu bytes of scratch, the static array holds %zu "
                                       "(GCMCRT_STATIC_SCRATCH_BYTES): pass fewer channels per call", ncr, ncol, need, kStaticScratchBytes);
        return fail(g, GCMCRT_E_INVALID, msg);
    }
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    void* base = nullptr;
    CUDA_TRY(g, static_scratch_address(&base));
    double* col_tot = static_cast<double*>(base);
    double* tot = col_tot + size_t(ncr) * ncol;
    const bool odev = is_device_ptr(L_tot);
    const GeomParams gp = geom_params(g);
    EmisParams ep;
    std::memset(static_cast<void*>(&ep), 0, sizeof ep);
    ep.n_chan = ncr; ep.nlev = g->nlev; ep.nlat = g->nlat; ep.nlon = g->nlon; ep.ncell = g->ncell;
    ep.alpha = g->alpha.as<float>() + size_t(cb) * gp.alpha_stride;
    ep.prop = g->prop.as<float4>() + size_t(cb) * g->ncell;
    ep.alpha_stride = gp.alpha_stride; ep.col_stride = gp.col_stride;
    ep.rho = g->rho.as<float>(); ep.T = g->T.as<float>();
    ep.lambda = g->lambda64.as<double>() + cb;
    ep.r_edges = g->r64.as<double>(); ep.cth_edges = g->cth64.as<double>(); ep.ph_edges = g->ph64.as<double>();
    ep.tau_vert_max = tau_vert_max;
    const int wpb = kEmisThreads / 32;
    const dim3 ge((unsigned)std::min((ncol + wpb - 1) / wpb, 32), (unsigned)std::min(ncr, 65535));
    const size_t sm = 2 * size_t(g->nlev) * sizeof(double);   // <= 4 KB: no attribute to set
    // nothing in the scratch has to start at zero: every entry that is read below is written by this call first
    if (g->nlev <= 64) emis_coltot_static_kernel<2><<<ge, kEmisThreads, sm, s>>>(ep, col_tot);
    else if (g->nlev <= 128) emis_coltot_static_kernel<4><<<ge, kEmisThreads, sm, s>>>(ep, col_tot);
    else emis_coltot_static_kernel<8><<<ge, kEmisThreads, sm, s>>>(ep, col_tot);
    CUDA_TRY(g, cudaGetLastError());
    // the column totals are added in column order by the kernel gcmcrt_run_emission uses (it leaves the exclusive sums
    // in col_tot, which nobody reads here)
    emis_colscan_kernel<<<(unsigned)((size_t(ncr) * 32 + 127) / 128), 128, 0, s>>>(ncr, ncol, col_tot, odev ? L_tot : tot);
    CUDA_TRY(g, cudaGetLastError());
    if (!odev) {
        CUDA_TRY(g, cudaMemcpyAsync(L_tot, tot, size_t(ncr) * sizeof(double), cudaMemcpyDeviceToHost, s));
        CUDA_TRY(g, cudaStreamSynchronize(s));
    }
    return GCMCRT_OK;
}

}  // extern "C"

// manta_api.cu -- host side of libmanta.so: the C ABI of include/manta.h.
// Initialisation (manta_create, manta_load_trips) validates, lays out the atlas / route store / queues and uploads;
// manta_step only enqueues kernels.  No simulator arithmetic runs on the host.
#include "../../include/manta.h"
#include "manta_kernels.cuh"

#include <algorithm>
#include <atomic>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <numeric>
#include <string>
#include <chrono>
#include <thread>
#include <vector>

using namespace manta;

// Scratch of manta_readback_noalloc (include/manta.h): the per-trip staging arrays that manta_readback takes from the
// allocator live here instead, in device memory that belongs to the loaded library itself.  Every device that loads
// libmanta.so holds these 7 MiB until the process exits.  In HOST code the name below is only a handle for
// cudaGetSymbolAddress -- it is not a device address and must never be handed to a kernel or a memset as one.
#define MANTA_NOALLOC_BYTES_PER_TRIP 28u   /* results 8 | route_pos 4 | x 4 | v 4 | acc 4 | status, lane, tag, wait 1 each */
#define MANTA_NOALLOC_SCRATCH_BYTES ((uint64_t)MANTA_NOALLOC_MAX_TRIPS * MANTA_NOALLOC_BYTES_PER_TRIP + 256u)
static __device__ __align__(256) unsigned char g_noalloc_scratch[MANTA_NOALLOC_SCRATCH_BYTES];

namespace {

manta_alloc_fn g_alloc = nullptr;
manta_free_fn g_free = nullptr;
void *g_alloc_ctx = nullptr;
cudaStream_t g_default_stream = 0;   // manta_set_default_stream: stream of the simulations created afterwards
thread_local std::string g_last_error;

struct Alloc {
    void *p;
    uint64_t bytes;
};

}  // namespace

struct manta_sim {
    int device = 0;
    cudaStream_t stream = 0;
    manta_params prm{};
    DevP P{};
    std::string err;
    bool sticky_cuda = false;
    std::vector<Alloc> allocs;
    uint64_t dev_bytes = 0, launches = 0;
    // host copies of the network
    uint32_t n_nodes = 0, n_edges = 0;
    std::vector<uint32_t> row_ptr, head, tail, len_c, cell_off;
    std::vector<uint8_t> lanes, node_prio;   // node_prio: the node is PRIORITY or STOP (one vehicle per step: the claim word is the node)
    bool has_stop = false;
    uint32_t min_len_c = 0;
    bool fuse_admit = false;      // admission of step t + 1 runs inside the second phase of step t (two barriers per step)
    double max_limit = 0.0;
    uint64_t n_cells = 0;
    // trips
    uint32_t n_trips = 0;
    bool loaded = false;
    uint32_t *d_trip_of_id = nullptr;
    uint32_t t = 0;
    int sm_count = 148;
    int grid_step = 1, grid_admit = 1, grid_persist = 0;   // blocks of the segment kernels / admission / persistent kernel
    bool w256 = true;             // look-ahead <= 256 cells and look-back <= 128: whole-window scans
    void *l2_window_base = nullptr;   // occupancy planes: L2 access-policy window of the step kernels
    uint64_t l2_window_bytes = 0;
    size_t l2_want = 0;               // carve-out the two planes would need (0: they do not fit, or MANTA_FLAG_NO_L2_PIN)
    size_t l2_persist = 0;            // persisting L2 carve-out currently granted (0 = not pinned now)
    uint64_t live_slots = 0;          // vehicle slots in use at the last manta_sync / manta_load_trips / manta_load_state: decides whether pinning pays (pin_update)
    std::vector<uint32_t> seg_cnt_host;   // manta_sync's copy of the segment counts
    uint32_t n_blk_stats = 0;
};

namespace {

int fail(manta_sim *s, int code, const char *fmt, ...)
{
    char buf[512];
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(buf, sizeof buf, fmt, ap);
    va_end(ap);
    g_last_error = buf;
    if (s) s->err = buf;
    return code;
}

#define CUDA_TRY(s, expr)                                                                          \
    do {                                                                                           \
        cudaError_t e_ = (expr);                                                                   \
        if (e_ != cudaSuccess) {                                                                   \
            if (s) (s)->sticky_cuda = true;                                                        \
            return fail(s, e_ == cudaErrorMemoryAllocation ? MANTA_ERR_OOM : MANTA_ERR_CUDA,       \
                        "%s: %s", #expr, cudaGetErrorString(e_));                                  \
        }                                                                                          \
    } while (0)

void *dev_alloc(manta_sim *s, uint64_t bytes)
{
    if (bytes == 0) bytes = 16;
    void *p = nullptr;
    if (g_alloc)
        p = g_alloc(bytes, s->device, g_alloc_ctx);
    else if (cudaMalloc(&p, bytes) != cudaSuccess) {
        cudaGetLastError();
        p = nullptr;
    }
    if (p) {
        s->allocs.push_back({p, bytes});
        s->dev_bytes += bytes;
    }
    return p;
}
void dev_free(manta_sim *s, void *p)
{
    for (size_t i = 0; i < s->allocs.size(); i++)
        if (s->allocs[i].p == p) {
            s->dev_bytes -= s->allocs[i].bytes;
            s->allocs.erase(s->allocs.begin() + (long)i);
            break;
        }
    if (g_free)
        g_free(p, s->device, g_alloc_ctx);
    else if (!g_alloc)
        cudaFree(p);
}

template <class T>
int upload(manta_sim *s, T **dst, const T *src, uint64_t n)
{
    *dst = (T *)dev_alloc(s, n * sizeof(T));
    if (!*dst) return fail(s, MANTA_ERR_OOM, "device allocation of %llu bytes failed", (unsigned long long)(n * sizeof(T)));
    if (n) CUDA_TRY(s, cudaMemcpyAsync(*dst, src, n * sizeof(T), cudaMemcpyHostToDevice, s->stream));
    return MANTA_OK;
}
template <class T>
int alloc_fill(manta_sim *s, T **dst, uint64_t n, int byte)
{
    *dst = (T *)dev_alloc(s, n * sizeof(T));
    if (!*dst) return fail(s, MANTA_ERR_OOM, "device allocation of %llu bytes failed", (unsigned long long)(n * sizeof(T)));
    CUDA_TRY(s, cudaMemsetAsync(*dst, byte, std::max<uint64_t>(n * sizeof(T), 1), s->stream));
    return MANTA_OK;
}

// R0 constants that depend on the fastest possible vehicle
void derive_constants(manta_sim *s, double max_init_speed)
{
    const manta_params &p = s->prm;
    // the fastest possible vehicle: the largest desired speed (3/2 of the largest limit with per-driver v0, R3s)
    const double vmax = s->max_limit * (p.v0_sigma_rel > 0.f ? 1.5 : 1.0);
    const double vcap = std::max(vmax, max_init_speed) + (double)p.a * (double)p.dt;
    s->P.L_c = (uint32_t)std::ceil((double)p.veh_len);
    s->P.L_fx = (int32_t)std::lround((double)p.veh_len * 1024.0);
    s->P.Z_out = (uint32_t)std::ceil(vcap * (double)p.dt) + 1u;
    s->P.Z_in = s->P.L_c + s->P.Z_out;
    float vc = (float)vcap;
    if ((double)vc < vcap) vc = std::nextafterf(vc, INFINITY);   // rounded up: the bound manta_load_state holds speeds to
    s->P.vcap = vc;
}
uint32_t len_min(const manta_sim *s) { return std::max(s->P.Z_out + 1u, s->P.L_c + 1u); }

// Stable counting sort on several host threads: out[r] = i for the r-th element in (key[i], i) order; elements with
// key == MANTA_NONE are left out.  start[k] (size n_keys + 1) receives the offset of key k's run.  Every thread
// counts its own contiguous range of i, the offsets are interleaved (key-major, thread-minor), every thread scatters
// its range: ranges are in index order, so the order inside a key's run is the index order.
void counting_sort_stable(const uint32_t *key, uint32_t n, uint32_t n_keys, std::vector<uint32_t> &start, std::vector<uint32_t> &out)
{
    const unsigned hw = std::max(1u, std::thread::hardware_concurrency());
    unsigned nt = n < (1u << 18) ? 1u : std::min(hw, 8u);
    while (nt > 1u && (uint64_t)nt * n_keys > (48ull << 20)) nt /= 2u;   // bound the per-thread histograms
    std::vector<uint32_t> hist((size_t)nt * n_keys, 0u);
    auto range = [&](unsigned w, uint64_t &i0, uint64_t &i1) { i0 = (uint64_t)n * w / nt; i1 = (uint64_t)n * (w + 1) / nt; };
    auto run = [&](auto fn) {
        if (nt == 1u) { fn(0u); return; }
        std::vector<std::thread> th;
        for (unsigned w = 0; w < nt; w++) th.emplace_back([=, &fn] { fn(w); });
        for (auto &t : th) t.join();
    };
    run([&](unsigned w) {
        uint64_t i0, i1;
        range(w, i0, i1);
        uint32_t *h = hist.data() + (size_t)w * n_keys;
        for (uint64_t i = i0; i < i1; i++)
            if (key[i] != MANTA_NONE) h[key[i]]++;
    });
    start.assign((size_t)n_keys + 1, 0u);
    uint32_t acc = 0u;
    for (uint32_t k = 0; k < n_keys; k++) {
        start[k] = acc;
        for (unsigned w = 0; w < nt; w++) {
            uint32_t &h = hist[(size_t)w * n_keys + k];
            const uint32_t c = h;
            h = acc;
            acc += c;
        }
    }
    start[n_keys] = acc;
    out.resize(acc);
    run([&](unsigned w) {
        uint64_t i0, i1;
        range(w, i0, i1);
        uint32_t *h = hist.data() + (size_t)w * n_keys;
        for (uint64_t i = i0; i < i1; i++)
            if (key[i] != MANTA_NONE) out[h[key[i]]++] = (uint32_t)i;
    });
}

// fn(i0, i1) over [0, n) in contiguous ranges on up to 16 host threads (small n: the calling thread alone)
template <class F>
void parallel_ranges(uint64_t n, F fn)
{
    const unsigned hw = std::max(1u, std::thread::hardware_concurrency());
    const unsigned nt = n < (1ull << 18) ? 1u : std::min(hw, 16u);
    if (nt == 1u) {
        fn((uint64_t)0, n);
        return;
    }
    std::vector<std::thread> th;
    for (unsigned w = 0; w < nt; w++) th.emplace_back([=, &fn] { fn(n * w / nt, n * (w + 1) / nt); });
    for (auto &t : th) t.join();
}

}  // namespace

extern "C" {

int manta_set_allocator(manta_alloc_fn alloc, manta_free_fn free_, void *ctx)
{
    if ((alloc == nullptr) != (free_ == nullptr)) return fail(nullptr, MANTA_ERR_INVALID_ARG, "allocator needs both callbacks");
    g_alloc = alloc;
    g_free = free_;
    g_alloc_ctx = ctx;
    return MANTA_OK;
}

const char *manta_last_error(const manta_sim *sim) { return sim ? sim->err.c_str() : g_last_error.c_str(); }
uint64_t manta_launch_count(const manta_sim *sim) { return sim ? sim->launches : 0; }
uint64_t manta_device_bytes(const manta_sim *sim) { return sim ? sim->dev_bytes : 0; }
uint64_t manta_atlas_cells(const manta_sim *sim) { return sim ? sim->n_cells : 0; }

namespace { void pin_release(manta_sim *s); }
void manta_destroy(manta_sim *sim)
{
    if (!sim) return;
    cudaSetDevice(sim->device);
    cudaStreamSynchronize(sim->stream);
    while (!sim->allocs.empty()) dev_free(sim, sim->allocs.back().p);
    if (sim->l2_persist) pin_release(sim);
    delete sim;
}

int manta_set_default_stream(void *cuda_stream)
{
    g_default_stream = (cudaStream_t)cuda_stream;
    return MANTA_OK;
}

int manta_set_stream(manta_sim *sim, void *cuda_stream)
{
    if (!sim) return fail(nullptr, MANTA_ERR_INVALID_ARG, "null simulation");
    sim->stream = (cudaStream_t)cuda_stream;
    return MANTA_OK;
}

int manta_set_multi_kernel(manta_sim *sim, int on)
{
    if (!sim) return fail(nullptr, MANTA_ERR_INVALID_ARG, "null simulation");
    if (on)
        sim->prm.flags |= MANTA_FLAG_MULTI_KERNEL;
    else
        sim->prm.flags &= ~MANTA_FLAG_MULTI_KERNEL;
    return MANTA_OK;
}

int manta_create(const manta_network *net, const manta_params *prm, int cuda_device, manta_sim **out)
{
    if (!net || !prm || !out) return fail(nullptr, MANTA_ERR_INVALID_ARG, "null argument");
    *out = nullptr;
    if (prm->size != sizeof(manta_params)) return fail(nullptr, MANTA_ERR_INVALID_ARG, "manta_params.size mismatch");
    if (!net->row_ptr || !net->head || !net->length_m || !net->lanes || !net->speed_limit || net->n_nodes == 0 ||
        net->n_edges == 0)
        return fail(nullptr, MANTA_ERR_INVALID_ARG, "network arrays missing");
    const manta_params &p = *prm;
    if (!(p.dt > 0.f) || !(p.a > 0.f) || !(p.b > 0.f) || !(p.T >= 0.f) || !(p.s0 >= 0.f) || !(p.veh_len > 0.f) ||
        !(p.veh_len <= 62.f) ||   // the entry window [0, L_c] of R1 is tested in one 64-cell word
        p.lookahead_cells < 1 || p.lookahead_cells > 8192 || p.lookback_cells < 1 || p.lookback_cells > 8192 ||
        !(p.mlc_scale_m >= 1.f) || !(p.mlc_scale_m <= 10000.f) || !(p.lc_alpha >= 0.f) || !(p.lc_eps_sigma >= 0.f) ||
        !std::isfinite(p.dlc_gain_thr) || !std::isfinite(p.lc_gap_low) || !std::isfinite(p.lc_gap_high) ||
        !(p.stop_time_s >= 0.f) || !std::isfinite(p.stop_time_s) ||   // (its length in steps is limited only where STOP nodes exist: below)
        !(p.v0_sigma_rel >= 0.f) || !std::isfinite(p.v0_sigma_rel) ||
        (p.stat_period_steps != 0u && (p.stat_slice_steps == 0u || p.stat_n_slices == 0u || p.stat_n_slices > 4096u)))
        return fail(nullptr, MANTA_ERR_INVALID_ARG, "parameter out of range");
    int n_dev = 0;
    if (cudaGetDeviceCount(&n_dev) != cudaSuccess || cuda_device < 0 || cuda_device >= n_dev) {
        cudaGetLastError();
        return fail(nullptr, MANTA_ERR_CUDA, "no CUDA device %d (there is no CPU fallback)", cuda_device);
    }
    manta_sim *s = new manta_sim();
    s->device = cuda_device;
    s->stream = g_default_stream;
    s->prm = p;
    auto bail = [&](int rc) {
        std::string e = s->err;
        manta_destroy(s);
        g_last_error = e;
        return rc;
    };
    if (cudaSetDevice(cuda_device) != cudaSuccess) return bail(fail(s, MANTA_ERR_CUDA, "cudaSetDevice failed"));
    cudaDeviceGetAttribute(&s->sm_count, cudaDevAttrMultiProcessorCount, cuda_device);

    // ---- validate + lay out the atlas (one row of 1 m cells per road lane)
    const uint32_t N = net->n_nodes, M = net->n_edges;
    s->n_nodes = N;
    s->n_edges = M;
    if (net->row_ptr[0] != 0 || net->row_ptr[N] != M) return bail(fail(s, MANTA_ERR_BAD_NETWORK, "row_ptr does not span the edges"));
    // packing limits of the device records: a node id is kept in 27 bits (NODE_MASK), lane entries
    // (e * 8 + lane) and claim-word indices (n_edges * 8 + node) are 32-bit
    static_assert(MANTA_MAX_LANES <= 8, "lane entries are e * 8 + lane");
    // (bit 27 of the node word in edge_tab.z / S3.z is the STOP flag in every network, so node ids stay below 2^27)
    if (N >= (1u << 27) || (uint64_t)M * 8ull + (uint64_t)N >= 0xFFFFFFFFull)
        return bail(fail(s, MANTA_ERR_BAD_NETWORK, "network too large for the device records (n_nodes < 2^27, 8 n_edges + n_nodes < 2^32)"));
    s->row_ptr.assign(net->row_ptr, net->row_ptr + N + 1);
    s->head.assign(net->head, net->head + M);
    s->tail.resize(M);
    s->lanes.assign(net->lanes, net->lanes + M);
    s->len_c.resize(M);
    s->cell_off.resize(M);
    for (uint32_t u = 0; u < N; u++) {
        if (s->row_ptr[u + 1] < s->row_ptr[u]) return bail(fail(s, MANTA_ERR_BAD_NETWORK, "row_ptr not monotone at node %u", u));
        if (s->row_ptr[u + 1] - s->row_ptr[u] > 255u) return bail(fail(s, MANTA_ERR_BAD_NETWORK, "out-degree of node %u > 255", u));
        for (uint32_t e = s->row_ptr[u]; e < s->row_ptr[u + 1]; e++) s->tail[e] = u;
    }
    s->max_limit = 0.0;
    uint64_t cells = 0;
    for (uint32_t e = 0; e < M; e++) {
        const float L = net->length_m[e], lim = net->speed_limit[e];
        if (!(net->lanes[e] >= 1 && net->lanes[e] <= MANTA_MAX_LANES) || !std::isfinite(L) || !(L > 0.f) ||
            !std::isfinite(lim) || !(lim > 0.f) || net->head[e] >= N)
            return bail(fail(s, MANTA_ERR_BAD_NETWORK, "edge %u: bad lanes / length / limit / head", e));
        const long lc = std::lround((double)L);
        if (lc > (long)MANTA_MAX_EDGE_CELLS) return bail(fail(s, MANTA_ERR_BAD_NETWORK, "edge %u longer than %u cells", e, MANTA_MAX_EDGE_CELLS));
        s->len_c[e] = (uint32_t)lc;
        s->max_limit = std::max(s->max_limit, (double)lim);
        if (cells > 0xFFFFFFFFull) return bail(fail(s, MANTA_ERR_BAD_NETWORK, "atlas exceeds 2^32 cells"));
        s->cell_off[e] = (uint32_t)cells;
        cells += (uint64_t)(((uint32_t)lc + 63u) & ~63u) * net->lanes[e];
    }
    if (cells + 256 > 0xFFFFFFFFull) return bail(fail(s, MANTA_ERR_BAD_NETWORK, "atlas exceeds 2^32 cells"));
    s->n_cells = cells;
    derive_constants(s, 0.0);
    for (uint32_t e = 0; e < M; e++)
        if (s->len_c[e] < len_min(s))
            return bail(fail(s, MANTA_ERR_BAD_NETWORK, "edge %u has %u cells < LEN_MIN %u (G19)", e, s->len_c[e], len_min(s)));

    // ---- constants of R0, rounded once from double
    DevP &P = s->P;
    P.dt = p.dt; P.a = p.a; P.T = p.T; P.s0 = p.s0; P.veh_len = p.veh_len;
    P.C1 = (float)(1.0 / (2.0 * std::sqrt((double)p.a * (double)p.b)));
    P.HALF_DT = (float)(0.5 * (double)p.dt);
    P.VSCALE = (float)((1.0 / 1024.0) / (double)p.dt);
    P.ADT = (float)((double)p.a * (double)p.dt);
    P.dlc_thr = p.dlc_gain_thr; P.alpha = p.lc_alpha; P.gap_low = p.lc_gap_low; P.gap_high = p.lc_gap_high;
    P.eps_sigma = p.lc_eps_sigma;
    P.H = p.lookahead_cells; P.lookback = p.lookback_cells;
    P.Lam = std::max<uint32_t>(1u, (uint32_t)std::lround((double)p.mlc_scale_m));
    P.seed_lo = (uint32_t)p.seed; P.seed_hi = (uint32_t)(p.seed >> 32);
    P.n_edges = M; P.flags = p.flags;

    s->node_prio.assign(N, 0);
    if (net->node_ctrl)
        for (uint32_t u = 0; u < N; u++) {
            if (net->node_ctrl[u] > MANTA_STOP) return bail(fail(s, MANTA_ERR_BAD_NETWORK, "node_ctrl value > 2 at node %u", u));
            s->node_prio[u] = net->node_ctrl[u] != MANTA_GREEN ? 1 : 0;
            s->has_stop = s->has_stop || net->node_ctrl[u] == MANTA_STOP;
        }
    const double w_stop = std::ceil((double)p.stop_time_s / (double)p.dt - 1e-9);
    if (s->has_stop && !(w_stop <= 7.0))   // only networks with STOP nodes use the 3-bit stop-line counter of S0.x
        return bail(fail(s, MANTA_ERR_INVALID_ARG, "stop_time_s = %g s is %.0f steps of dt = %g s; MANTA_STOP nodes allow at most 7 steps (3-bit stop-line counter)",
                         (double)p.stop_time_s, w_stop, (double)p.dt));
    P.W_stop = s->has_stop ? (uint32_t)w_stop : 0u;
    P.id_mask = s->has_stop ? 0x00FFFFFFu : 0xFFFFFFFFu;
    P.v0_sigma_rel = p.v0_sigma_rel;
    P.stat_period = p.stat_period_steps; P.stat_slice = p.stat_slice_steps; P.stat_n_slices = p.stat_period_steps ? p.stat_n_slices : 0u;
    s->min_len_c = *std::min_element(s->len_c.begin(), s->len_c.end());
    // ---- device tables
    std::vector<uint4> et(M);
    std::vector<uint4> es(s->has_stop ? M : 1u, make_uint4(0u, 0u, 0u, 0u));   // STOP nodes (R8s): {n_in * n_out, in_idx * n_out, first out-edge, 0}
    std::vector<uint32_t> indeg(N, 0u);
    for (uint32_t e = 0; e < M; e++) {
        const uint32_t u = s->head[e];
        const uint32_t prio = s->node_prio[u];
        const bool stop = net->node_ctrl && net->node_ctrl[u] == MANTA_STOP;
        uint32_t vb;
        memcpy(&vb, &net->speed_limit[e], 4);
        et[e] = make_uint4(s->cell_off[e], s->len_c[e] | ((uint32_t)s->lanes[e] << 16) | (prio << 27), u | (stop ? 1u << 27 : 0u), vb);
        if (stop) es[e].y = indeg[u];   // index among the node's inbound edges, in edge-id order (times n_out below)
        indeg[u]++;
    }
    if (s->has_stop)
        for (uint32_t e = 0; e < M; e++) {
            const uint32_t u = s->head[e];
            if (!(net->node_ctrl[u] == MANTA_STOP)) continue;
            const uint32_t m = s->row_ptr[u + 1] - s->row_ptr[u];
            if ((uint64_t)indeg[u] * m > 256u) return bail(fail(s, MANTA_ERR_BAD_NETWORK, "STOP node %u: in-degree x out-degree > 256", u));
            es[e] = make_uint4(indeg[u] * m, es[e].y * m, s->row_ptr[u], 0u);
        }
    std::vector<uint32_t> pm(5 * P.Lam + 1);
    for (uint32_t d = 0; d <= 5 * P.Lam; d++) {  // Eq. (2), distances in units of Lambda (G6)
        if (d <= P.Lam)
            pm[d] = 0xFFFFFFFFu;
        else {
            const double xi = (double)d / (double)P.Lam;
            pm[d] = (uint32_t)std::floor(4294967296.0 * std::exp(-(xi - 1.0) * (xi - 1.0)));
        }
    }
    int rc;
    uint4 *d_et; uint32_t *d_pm, *d_ee; u64 *d_claim; Counters *d_ctr; BlockStats *d_blk;
    if ((rc = upload(s, &d_et, et.data(), M))) return bail(rc);
    {
        uint4 *d_es;
        if ((rc = upload(s, &d_es, es.data(), es.size()))) return bail(rc);
        P.edge_stop = d_es;
    }
    if (P.stat_n_slices) {
        if ((rc = alloc_fill(s, &P.stat_sum, (uint64_t)P.stat_n_slices * M, 0))) return bail(rc);
        if ((rc = alloc_fill(s, &P.stat_cnt, (uint64_t)P.stat_n_slices * M, 0))) return bail(rc);
    }
    if ((rc = upload(s, &d_pm, pm.data(), pm.size()))) return bail(rc);
    if ((rc = alloc_fill(s, &d_ee, M, 0))) return bail(rc);
    if ((rc = alloc_fill(s, &d_claim, (uint64_t)M * 8 + N, 0xFF))) return bail(rc);
    if ((rc = alloc_fill(s, &d_ctr, 1, 0))) return bail(rc);
    s->n_blk_stats = (uint32_t)s->sm_count * 16u;
    if ((rc = alloc_fill(s, &d_blk, s->n_blk_stats, 0))) return bail(rc);
    {   // both occupancy planes in one allocation, so that one L2 access-policy window covers them
        const uint64_t plane_words = ((cells / 64 + 8) + 15) & ~15ull;
        u64 *planes;
        if ((rc = alloc_fill(s, &planes, 2 * plane_words, 0))) return bail(rc);
        P.bits[0] = planes;
        P.bits[1] = planes + plane_words;
        // The occupancy planes are the most re-read data of a step (every look-ahead reads them, every vehicle
        // toggles two marks); pin them in L2 so that the streamed state and payload sectors do not evict them.
        s->l2_window_base = planes;
        s->l2_window_bytes = 2 * plane_words * sizeof(u64);
        int max_persist = 0, max_window = 0;
        cudaDeviceGetAttribute(&max_persist, cudaDevAttrMaxPersistingL2CacheSize, cuda_device);
        cudaDeviceGetAttribute(&max_window, cudaDevAttrMaxAccessPolicyWindowSize, cuda_device);
        s->l2_persist = 0;
        // Only when both planes fit the carve-out and one window: a window larger than the carve-out leaves part of
        // its lines on the evict-first miss policy, which costs far more than it saves (configs[4], 178 MB of planes:
        // 400 us per step pinned, 142 us unpinned; profiles/r01d_*).
        if (!(p.flags & MANTA_FLAG_NO_L2_PIN) && max_persist > 0 && max_window > 0 &&
            s->l2_window_bytes <= (uint64_t)max_persist && s->l2_window_bytes <= (uint64_t)max_window) {
            s->l2_want = (size_t)std::min<uint64_t>(s->l2_window_bytes, (uint64_t)max_persist);
            s->l2_window_bytes = std::min<uint64_t>(s->l2_window_bytes, (uint64_t)max_window);
        }   // whether the window is USED is decided per manta_step call, by the load (pin_update)
    }
    P.pay_shift = P.L_fx >= 4096 ? 2u : 0u;   // one payload entry per aligned group of four cells when L >= 4 m
    for (int k = 0; k < 2; k++)
        if ((rc = alloc_fill(s, &P.pay[k], (cells >> P.pay_shift) + 64, 0))) return bail(rc);
    P.edge_tab = d_et; P.P_mlc = d_pm; P.edge_entries = d_ee; P.claim = d_claim; P.ctr = d_ctr;
    P.blk = d_blk;
    if (cudaStreamSynchronize(s->stream) != cudaSuccess) return bail(fail(s, MANTA_ERR_CUDA, "upload failed: %s", cudaGetErrorString(cudaGetLastError())));
    *out = s;
    return MANTA_OK;
}

int manta_load_trips(manta_sim *s, uint32_t n_trips, const uint64_t *route_ptr, const uint32_t *route_edges,
                     const float *depart_time_s, const float *init_pos_m, const float *init_speed)
{
    if (!s) return fail(nullptr, MANTA_ERR_INVALID_ARG, "null simulation");
    if (s->sticky_cuda) return fail(s, MANTA_ERR_CUDA, "earlier CUDA failure");
    if (s->loaded) return fail(s, MANTA_ERR_STATE, "trips already loaded");
    if (!route_ptr || !route_edges || !depart_time_s || n_trips == 0 || n_trips >= 0x7FFFFFFFu)
        return fail(s, MANTA_ERR_INVALID_ARG, "null / empty / too many trips");
    if (s->has_stop && n_trips >= (1u << 24))   // strictly: id 2^24 - 1 under turn rank 255 would give the key of an unclaimed word
        return fail(s, MANTA_ERR_INVALID_ARG, "networks with STOP nodes take fewer than 2^24 trips (the claim key keeps the turn rank above a 24-bit vehicle id)");
    CUDA_TRY(s, cudaSetDevice(s->device));
    // MANTA_LOAD_TIMING=1: wall time of each stage of this call on stderr (initialisation is outside the timed path,
    // but it is most of the end-to-end time of a short run)
    const bool timing = getenv("MANTA_LOAD_TIMING") != nullptr;
    auto t_prev = std::chrono::steady_clock::now();
    auto lap = [&](const char *what) {
        if (!timing) return;
        const auto now = std::chrono::steady_clock::now();
        fprintf(stderr, "[manta_load_trips] %-28s %8.2f ms\n", what, std::chrono::duration<double, std::milli>(now - t_prev).count());
        t_prev = now;
    };
    const uint64_t total = route_ptr[n_trips];
    if (route_ptr[0] != 0 || total >= 0xFFFFFFFFull) return fail(s, MANTA_ERR_BAD_ROUTE, "route_ptr must start at 0 and stay below 2^32 entries");
    // ---- validation (BAD_ROUTE): every route entry is looked at once; split over host threads for large inputs, the
    // error reported is that of the lowest trip index, as a sequential scan would report it
    // The route entries (by far the largest input: 0.8 GB at configs[2]) start their way to the device NOW, on a helper
    // thread, while this thread and its workers validate them and build ids and queues on the host: a copy from
    // pageable memory is staged by the driver and costs as much wall time as the validation.  If the validation
    // fails the copy is awaited and the buffer released.
    uint32_t *d_re = (uint32_t *)dev_alloc(s, total * sizeof(uint32_t));
    if (!d_re) return fail(s, MANTA_ERR_OOM, "device allocation of %llu bytes failed", (unsigned long long)(total * sizeof(uint32_t)));
    struct Uploader {
        std::thread th;
        cudaError_t err = cudaSuccess;
        void join() { if (th.joinable()) th.join(); }
        ~Uploader() { join(); }
    } up;
    up.th = std::thread([&up, s, d_re, route_edges, total] {
        cudaError_t e = cudaSetDevice(s->device);
        const uint64_t slice = 16ull << 20;   // entries per copy
        for (uint64_t off = 0; off < total && e == cudaSuccess; off += slice)
            e = cudaMemcpyAsync(d_re + off, route_edges + off, std::min(slice, total - off) * sizeof(uint32_t), cudaMemcpyHostToDevice, s->stream);
        up.err = e;
    });
    auto drop_upload = [&](int rc) {
        up.join();
        cudaStreamSynchronize(s->stream);
        dev_free(s, d_re);
        return rc;
    };
    std::vector<uint32_t> first_edge(n_trips);   // filled by the validation pass (route_ptr is walked in trip order there)
    struct Bad { uint32_t trip; int kind; uint64_t pos; };   // kind 0: none
    auto scan = [&](uint32_t i0, uint32_t i1, Bad &bad, double &max_init) {
        for (uint32_t i = i0; i < i1; i++) {
            const uint64_t b = route_ptr[i], e = route_ptr[i + 1];
            if (e <= b || e > total) { bad = {i, 1, 0}; return; }
            first_edge[i] = route_edges[b];
            for (uint64_t k = b; k < e; k++) {
                if (route_edges[k] >= s->n_edges) { bad = {i, 2, k - b}; return; }
                if (k > b && s->head[route_edges[k - 1]] != s->tail[route_edges[k]]) { bad = {i, 3, k - b}; return; }
            }
            const bool pre = init_pos_m && init_pos_m[i] >= 0.0f;
            if (!pre && !(depart_time_s[i] >= 0.0f)) { bad = {i, 4, 0}; return; }
            if (init_speed) {
                if (!(init_speed[i] >= 0.0f) || !std::isfinite(init_speed[i])) { bad = {i, 5, 0}; return; }
                if (pre) max_init = std::max(max_init, (double)init_speed[i]);
            }
        }
    };
    double max_init = 0.0;
    const unsigned hw_val = std::max(1u, std::thread::hardware_concurrency());
    const unsigned nt_val = total < (1ull << 20) ? 1u : std::min(hw_val, 32u);
    std::vector<Bad> bad(nt_val, Bad{0u, 0, 0});
    std::vector<double> mx(nt_val, 0.0);
    std::vector<std::thread> val_threads;   // large inputs: the workers run while this thread builds the vehicle ids
    if (nt_val == 1u) {
        scan(0u, n_trips, bad[0], mx[0]);
    } else {
        for (unsigned w = 0; w < nt_val; w++) {
            const uint32_t a = (uint32_t)((uint64_t)n_trips * w / nt_val), b = (uint32_t)((uint64_t)n_trips * (w + 1) / nt_val);
            val_threads.emplace_back([&, w, a, b] { scan(a, b, bad[w], mx[w]); });
        }
    }
    // ---- vehicle ids: rank in the stable (depart_step, trip index) order (needs only the departure times)
    std::vector<uint32_t> dstep(n_trips), trip_of_id;
    std::atomic<uint32_t> too_late(MANTA_NONE);   // lowest trip index whose departure step does not fit 32 bits
    parallel_ranges(n_trips, [&](uint64_t a, uint64_t b) {
        for (uint64_t i = a; i < b; i++) {
            const bool pre = init_pos_m && init_pos_m[i] >= 0.0f;
            const double ds = std::floor((double)depart_time_s[i] / (double)s->prm.dt);
            if (!pre && !(ds < 4294967295.0)) {   // (also NaN / negative garbage: reported by the validation)
                if (ds >= 4294967295.0) {
                    uint32_t cur = too_late.load();
                    while ((uint32_t)i < cur && !too_late.compare_exchange_weak(cur, (uint32_t)i)) {}
                }
                dstep[i] = 0u;
                continue;
            }
            dstep[i] = (pre || ds < 0.0) ? 0u : (uint32_t)ds;
        }
    });
    {
        const uint32_t max_step = *std::max_element(dstep.begin(), dstep.end());
        if (max_step < (1u << 24)) {   // counting sort by departure step, trip order kept inside a step (stable)
            std::vector<uint32_t> start;
            counting_sort_stable(dstep.data(), n_trips, max_step + 1u, start, trip_of_id);
        } else {
            trip_of_id.resize(n_trips);
            std::iota(trip_of_id.begin(), trip_of_id.end(), 0u);
            std::stable_sort(trip_of_id.begin(), trip_of_id.end(), [&](uint32_t x, uint32_t y) { return dstep[x] < dstep[y]; });
        }
    }
    for (auto &t : val_threads) t.join();
    for (unsigned w = 0; w < nt_val; w++) {   // ranges are in trip order: the first bad one is the lowest trip index
        const Bad &b = bad[w];
        switch (b.kind) {
        case 0: break;
        case 1: return drop_upload(fail(s, MANTA_ERR_BAD_ROUTE, "trip %u: empty route", b.trip));
        case 2: return drop_upload(fail(s, MANTA_ERR_BAD_ROUTE, "trip %u: edge id out of range", b.trip));
        case 3: return drop_upload(fail(s, MANTA_ERR_BAD_ROUTE, "trip %u: route not connected at position %llu", b.trip, (unsigned long long)b.pos));
        case 4: return drop_upload(fail(s, MANTA_ERR_BAD_ROUTE, "trip %u: negative departure time", b.trip));
        default: return drop_upload(fail(s, MANTA_ERR_BAD_ROUTE, "trip %u: bad init_speed", b.trip));
        }
        max_init = std::max(max_init, mx[w]);
    }
    if (too_late.load() != MANTA_NONE) return drop_upload(fail(s, MANTA_ERR_BAD_ROUTE, "trip %u: departure too late", too_late.load()));
    lap("validate routes | vehicle ids");
    const DevP saved = s->P;
    derive_constants(s, max_init);
    bool upload_joined = false;
    auto rollback = [&](int rc) {
        s->P = saved;
        if (!upload_joined) drop_upload(rc);
        return rc;
    };
    for (uint32_t e = 0; e < s->n_edges; e++)
        if (s->len_c[e] < len_min(s)) return rollback(fail(s, MANTA_ERR_BAD_ROUTE, "edge %u shorter than LEN_MIN for the pre-placed speeds", e));
    if (s->prm.lookback_cells < s->P.L_c + s->P.Z_out)
        return rollback(fail(s, MANTA_ERR_INVALID_ARG, "lookback_cells %u < L_c + Z_out = %u (R5)", s->prm.lookback_cells, s->P.L_c + s->P.Z_out));

    std::vector<uint32_t> depart_by_id(n_trips), route_start(n_trips), first_by_id(n_trips);
    parallel_ranges(n_trips, [&](uint64_t i0, uint64_t i1) {
        for (uint64_t id = i0; id < i1; id++) {
            const uint32_t tr = trip_of_id[id];
            depart_by_id[id] = dstep[tr];
            route_start[id] = (uint32_t)route_ptr[tr];
            first_by_id[id] = (init_pos_m && init_pos_m[tr] >= 0.0f) ? MANTA_NONE : first_edge[tr];   // NONE: pre-placed, no queue
        }
    });
    // ---- pre-placed vehicles (R1, last sentence) and their spacing check
    std::vector<uint4> init_a0;
    {
        std::vector<std::pair<uint64_t, uint32_t>> keyx;
        for (uint32_t id = 0; id < n_trips; id++) {
            const uint32_t tr = trip_of_id[id];
            if (!(init_pos_m && init_pos_m[tr] >= 0.0f)) continue;
            const uint32_t e = route_edges[route_ptr[tr]];
            const long x = std::lround((double)init_pos_m[tr] * 1024.0);
            if (x < 0 || (uint64_t)x >= ((uint64_t)s->len_c[e] << 10)) return rollback(fail(s, MANTA_ERR_BAD_ROUTE, "trip %u: init_pos_m beyond its edge", tr));
            const float v = init_speed ? init_speed[tr] : 0.0f;
            uint32_t vb;
            memcpy(&vb, &v, 4);
            init_a0.push_back(make_uint4((uint32_t)x, vb, id, route_start[id]));
            keyx.push_back({((uint64_t)e << 32) | (uint64_t)x, id});
        }
        std::sort(keyx.begin(), keyx.end());
        for (size_t k = 1; k < keyx.size(); k++)
            if ((keyx[k].first >> 32) == (keyx[k - 1].first >> 32) &&
                (int64_t)(keyx[k].first & 0xFFFFFFFFull) - (int64_t)(keyx[k - 1].first & 0xFFFFFFFFull) < (int64_t)s->P.L_fx)
                return rollback(fail(s, MANTA_ERR_BAD_ROUTE, "pre-placed vehicles closer than L on edge %llu", (unsigned long long)(keyx[k].first >> 32)));
    }
    lap("ids -> depart / route start, pre-placed");
    // ---- admission FIFOs: waiting trips grouped by first edge, id order inside (G25)
    // q_ent = {vehicle id, depart_step, route cursor, depart_step of the next entry of the same queue or NONE}
    std::vector<uint32_t> q_edge, q_end;
    std::vector<uint4> q_ent, q_row, q_state;
    {
        std::vector<uint32_t> cnt, q_ids;   // waiting vehicle ids grouped by first edge, id order inside a group
        counting_sort_stable(first_by_id.data(), n_trips, s->n_edges, cnt, q_ids);
        q_ent.resize(q_ids.size() + 1);
        q_ent.back() = make_uint4(MANTA_NONE, MANTA_NONE, 0u, MANTA_NONE);
        parallel_ranges(q_ids.size(), [&](uint64_t k0, uint64_t k1) {
            for (uint64_t k = k0; k < k1; k++) {
                const uint32_t id = q_ids[k];
                const bool has_next = k + 1 < q_ids.size() && first_by_id[q_ids[k + 1]] == first_by_id[id];
                q_ent[k] = make_uint4(id, depart_by_id[id], route_start[id], has_next ? depart_by_id[q_ids[k + 1]] : MANTA_NONE);
            }
        });
        for (uint32_t e = 0; e < s->n_edges; e++)
            if (cnt[e + 1] > cnt[e]) {
                q_edge.push_back(e);
                q_end.push_back(cnt[e + 1]);
                const uint4 h = q_ent[cnt[e]];
                q_state.push_back(make_uint4(h.y, cnt[e], h.x, h.z));
            }
    }
    lap("admission queues");
    // ---- launch geometry and vehicle segments.  A segment is processed by one block per phase; the persistent
    // kernel needs all of its blocks co-resident (cooperative launch), so n_seg = that grid.
    s->w256 = s->prm.lookahead_cells <= 256u && s->prm.lookback_cells <= 128u;
    // fused admission (see admit_phase): a claim loser's mark (last cell of its row) must lie beyond the entry
    // window [0, L_c], and a winner's landing cell must fit the first occupancy word
    s->fuse_admit = !(s->prm.flags & MANTA_FLAG_NO_FUSE) && s->min_len_c >= s->P.L_c + 2u && s->P.Z_out <= 63u;
    {
        int occ = 0, coop = 0;
        if (MANTA_REC_BYTES) {   // the two-stage pass keeps per-thread records in dynamic shared memory (opt-in above 48 KB)
            CUDA_TRY(s, cudaFuncSetAttribute(k_persistent<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, MANTA_REC_BYTES));
            CUDA_TRY(s, cudaFuncSetAttribute(k_persistent<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, MANTA_REC_BYTES));
            CUDA_TRY(s, cudaFuncSetAttribute(k_update<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, MANTA_REC_BYTES));
            CUDA_TRY(s, cudaFuncSetAttribute(k_update<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, MANTA_REC_BYTES));
        }
        if (s->w256)
            CUDA_TRY(s, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_persistent<true>, MANTA_NT, MANTA_REC_BYTES));
        else
            CUDA_TRY(s, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_persistent<false>, MANTA_NT, MANTA_REC_BYTES));
        CUDA_TRY(s, cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, s->device));
        s->grid_persist = (coop && occ > 0) ? std::min<int>(s->sm_count * occ, (int)s->n_blk_stats) : 0;
        s->grid_step = s->grid_persist ? s->grid_persist : std::min<int>(s->sm_count * 2, (int)s->n_blk_stats);
        if (s->prm.flags & MANTA_FLAG_FEW_SEGMENTS) {   // test switch: two segments / two blocks
            s->grid_step = std::min(s->grid_step, 2);
            if (s->grid_persist) s->grid_persist = s->grid_step;
        }
    }
    DevP &P = s->P;
    P.n_seg = (uint32_t)s->grid_step;
    P.seg_cap = (n_trips + P.n_seg - 1u) / P.n_seg + 256u;
    const uint64_t cap = (uint64_t)P.n_seg * P.seg_cap;
    if (cap >= 0xFFFFFFFFull || P.seg_cap >= (1u << 28))   // list entries keep the slot in 28 bits (cross list) / 30 bits (deferred list)
        return rollback(fail(s, MANTA_ERR_INVALID_ARG, "too many trips for the segment layout"));
    // ---- upload; expand the route store on the device
    int rc;
    uint32_t *d_rowptr = nullptr, *d_rs, *d_adm, *d_arr, *d_qend;
    uint64_t *d_rp = nullptr;
    uint4 *d_route, *d_qent, *d_qrow, *d_qstate;
    for (size_t k = 0; k < q_edge.size(); k++) {
        const uint32_t e = q_edge[k];
        const uint32_t prio_word = s->node_prio[s->tail[e]] ? s->n_edges * 8u + s->tail[e] : MANTA_NONE;
        q_row.push_back(make_uint4(s->cell_off[e], s->len_c[e] | ((uint32_t)s->lanes[e] << 16), prio_word, e));
    }
    lap("launch geometry");
    up.join();   // the route entries are on their way (enqueued on the simulation's stream)
    if (up.err != cudaSuccess) {
        s->sticky_cuda = true;
        return rollback(fail(s, MANTA_ERR_CUDA, "route upload failed: %s", cudaGetErrorString(up.err)));
    }
    upload_joined = true;
    if ((rc = upload(s, &d_rp, route_ptr, (uint64_t)n_trips + 1))) return rollback(rc);
    if ((rc = upload(s, &d_rowptr, s->row_ptr.data(), s->row_ptr.size()))) return rollback(rc);
    d_route = (uint4 *)dev_alloc(s, (total + 8) * sizeof(uint4));   // + 8: the look-ahead requests four records ahead
    if (!d_route) return rollback(fail(s, MANTA_ERR_OOM, "route store allocation failed"));
    CUDA_TRY(s, cudaMemsetAsync(d_route + total, 0, 8 * sizeof(uint4), s->stream));
    k_expand_routes<<<(unsigned)std::min<uint64_t>((total + 255) / 256, 65535ull * 16), 256, 0, s->stream>>>(P.edge_tab, d_rowptr, d_re, total, d_route);
    k_mark_last<<<(n_trips + 255) / 256, 256, 0, s->stream>>>(d_rp, n_trips, d_route);
    CUDA_TRY(s, cudaGetLastError());
    lap("route upload + expand (enqueued)");
    if ((rc = upload(s, &d_rs, route_start.data(), n_trips))) return rollback(rc);
    if ((rc = upload(s, &s->d_trip_of_id, trip_of_id.data(), n_trips))) return rollback(rc);
    if ((rc = alloc_fill(s, &d_adm, n_trips, 0xFF))) return rollback(rc);
    if ((rc = alloc_fill(s, &d_arr, n_trips, 0xFF))) return rollback(rc);
    if ((rc = upload(s, &d_qrow, q_row.data(), q_row.size()))) return rollback(rc);
    if ((rc = upload(s, &d_qent, q_ent.data(), q_ent.size()))) return rollback(rc);
    if ((rc = upload(s, &d_qend, q_end.data(), q_end.size()))) return rollback(rc);
    if ((rc = upload(s, &d_qstate, q_state.data(), q_state.size()))) return rollback(rc);
    {   // for manta_load_state: where each queue starts, how long each route is
        std::vector<uint32_t> q_begin(q_state.size()), route_len(n_trips);
        for (size_t k = 0; k < q_state.size(); k++) q_begin[k] = q_state[k].y;
        parallel_ranges(n_trips, [&](uint64_t i0, uint64_t i1) {
            for (uint64_t id = i0; id < i1; id++) route_len[id] = (uint32_t)(route_ptr[trip_of_id[id] + 1] - route_ptr[trip_of_id[id]]);
        });
        uint32_t *d_qb, *d_rl;
        if ((rc = upload(s, &d_qb, q_begin.data(), q_begin.size()))) return rollback(rc);
        if ((rc = upload(s, &d_rl, route_len.data(), route_len.size()))) return rollback(rc);
        CUDA_TRY(s, cudaStreamSynchronize(s->stream));   // the vectors go out of scope
        P.q_begin = d_qb;
        P.route_len = d_rl;
    }
    if ((rc = alloc_fill(s, &P.cand_info, n_trips, 0))) return rollback(rc);
    for (int k = 0; k < 2; k++) {
        uint4 **arr[4] = {&P.st[k].S0, &P.st[k].S1, &P.st[k].S2, &P.st[k].S3};
        for (int a = 0; a < 4; a++) {
            *arr[a] = (uint4 *)dev_alloc(s, cap * sizeof(uint4));
            if (!*arr[a]) return rollback(fail(s, MANTA_ERR_OOM, "vehicle array allocation failed"));
        }
        P.st[k].acc = (s->prm.flags & MANTA_FLAG_RECORD_ACC) ? (float *)dev_alloc(s, cap * sizeof(float)) : nullptr;
        if (P.st[k].acc) CUDA_TRY(s, cudaMemsetAsync(P.st[k].acc, 0, cap * sizeof(float), s->stream));
    }
    if ((rc = alloc_fill(s, &P.seg_cnt, P.n_seg, 0))) return rollback(rc);
    {   // re-sort scratch; until the first sort admission spreads the origins evenly over the segments
        P.n_buckets = (uint32_t)((s->n_cells + (1ull << MANTA_BUCKET_SHIFT) - 1) >> MANTA_BUCKET_SHIFT) + 1u;
        if ((rc = alloc_fill(s, &P.sort_hist, (uint64_t)P.n_buckets + 1, 0))) return rollback(rc);
        if ((rc = alloc_fill(s, &P.sort_part, (uint64_t)P.n_seg + 2, 0))) return rollback(rc);
        if ((rc = alloc_fill(s, &P.sort_rank, cap, 0xFF))) return rollback(rc);
        std::vector<uint32_t> bs(P.n_buckets);
        for (uint32_t b = 0; b < P.n_buckets; b++) bs[b] = (uint32_t)(((uint64_t)b * P.n_seg) / P.n_buckets);
        if ((rc = upload(s, &P.bucket_seg, bs.data(), bs.size()))) return rollback(rc);
        CUDA_TRY(s, cudaStreamSynchronize(s->stream));   // bs goes out of scope
    }
    lap("tables, state arrays, sort scratch (sync)");
    if ((rc = alloc_fill(s, &P.seg_xn, P.n_seg, 0))) return rollback(rc);
    if ((rc = alloc_fill(s, &P.dbg_buf, (uint64_t)P.n_seg * 8, 0))) return rollback(rc);
    if ((rc = alloc_fill(s, &P.seg_qn, P.n_seg, 0))) return rollback(rc);
    P.xlist = (uint4 *)dev_alloc(s, cap * sizeof(uint4));
    P.dlist = (uint4 *)dev_alloc(s, cap * sizeof(uint4));
    if (!P.xlist || !P.dlist) return rollback(fail(s, MANTA_ERR_OOM, "vehicle array allocation failed"));
    P.route = d_route; P.route_start = d_rs; P.admit_step = d_adm; P.arrive_step = d_arr;
    P.q_row = d_qrow; P.q_ent = d_qent; P.q_end = d_qend; P.q_state = d_qstate;
    P.n_queues = (uint32_t)q_edge.size();
    const uint32_t n_init = (uint32_t)init_a0.size();
    if (n_init) {
        uint4 *d_init;
        if ((rc = upload(s, &d_init, init_a0.data(), n_init))) return rollback(rc);
        std::vector<uint32_t> cnt0(P.n_seg);
        for (uint32_t k = 0; k < P.n_seg; k++) cnt0[k] = n_init / P.n_seg + (k < n_init % P.n_seg ? 1u : 0u);
        CUDA_TRY(s, cudaMemcpyAsync(P.seg_cnt, cnt0.data(), (uint64_t)P.n_seg * 4, cudaMemcpyHostToDevice, s->stream));
        k_place_initial<<<(n_init + 255) / 256, 256, 0, s->stream>>>(P, d_init, n_init);
        CUDA_TRY(s, cudaGetLastError());
        CUDA_TRY(s, cudaStreamSynchronize(s->stream));
        dev_free(s, d_init);
    }
    CUDA_TRY(s, cudaStreamSynchronize(s->stream));
    dev_free(s, d_re);
    dev_free(s, d_rp);
    dev_free(s, d_rowptr);
    lap("lists, initial placement, final sync");
#ifdef MANTA_CHECK
    {   // sizes the device-side bounds checks compare against
        CheckCtx c{};
        c.plane_words = ((s->n_cells / 64 + 8) + 15) & ~15ull;
        c.pay_entries = (s->n_cells >> P.pay_shift) + 64;
        c.n_cells = s->n_cells;
        c.n_claims = (uint64_t)s->n_edges * 8 + s->n_nodes;
        c.route_total = total;
        c.slots = cap;
        c.n_edges = s->n_edges;
        c.n_trips = n_trips;
        c.fail = 0;
        CUDA_TRY(s, cudaMemcpyToSymbol(g_check, &c, sizeof c));
    }
#endif
    s->n_trips = n_trips;
    s->loaded = true;
    s->t = 0;
    s->live_slots = n_init;   // slots in use before the first step: the pre-placed vehicles
    s->grid_admit = (int)std::max<uint32_t>(1u, std::min<uint32_t>((P.n_queues + 255u) / 256u, (uint32_t)s->sm_count * 8u));   // k_admit alone
    return MANTA_OK;
}

namespace {

int check_ready(manta_sim *s, uint32_t n_steps)
{
    if (!s) return fail(nullptr, MANTA_ERR_INVALID_ARG, "null simulation");
    if (s->sticky_cuda) return fail(s, MANTA_ERR_CUDA, "earlier CUDA failure");
    if (!s->loaded) return fail(s, MANTA_ERR_STATE, "no trips loaded");
    if ((uint64_t)s->t + n_steps >= 0xFFFFFFFEull) return fail(s, MANTA_ERR_INVALID_ARG, "step counter would overflow");
    return MANTA_OK;
}

// The persisting carve-out takes L2 away from everything else.  It pays once the touched working set of a step no
// longer fits L2 next to the planes: measured at configs[2] / [3] (profiles/r02_final.md), pinned vs not: 26.3 vs 24.7 us
// per step at 0.29 M vehicles, 30.6 vs 30.7 at 0.45 M, 40.0 vs 40.5 at 0.67 M, 84.2 vs 86.3 at 2.1 M.  So the window is
// switched on for a manta_step call that starts with at least MANTA_PIN_MIN_SLOTS vehicle slots in use (as counted at
// the last manta_sync) and off below (the decision holds for the whole call: the host is not involved between steps).
// cudaLimitPersistingL2CacheSize is a device-wide setting: raised while pinning, put back afterwards.
#ifndef MANTA_PIN_MIN_SLOTS
#define MANTA_PIN_MIN_SLOTS 400000ull
#endif
// Several simulations may pin on one device (replica runs, batches): the limit found before the FIRST of them pinned is
// kept per device and put back, and the persisting lines reset, only when the LAST pinned one lets go.
struct PinDevice {
    int pinned = 0;            // simulations on this device that hold a window now
    size_t original = 0;       // cudaLimitPersistingL2CacheSize before the first of them
    bool raised = false;       // the library raised the limit above `original`
};
std::mutex g_pin_mu;
PinDevice g_pin[64];

bool pin_acquire(manta_sim *s)   // device current
{
    if (s->device < 0 || s->device >= 64) return false;
    std::lock_guard<std::mutex> lock(g_pin_mu);
    PinDevice &d = g_pin[s->device];
    size_t now = 0;
    if (cudaDeviceGetLimit(&now, cudaLimitPersistingL2CacheSize) != cudaSuccess) { cudaGetLastError(); return false; }
    if (d.pinned == 0) { d.original = now; d.raised = false; }
    if (now < s->l2_want) {
        if (cudaDeviceSetLimit(cudaLimitPersistingL2CacheSize, s->l2_want) != cudaSuccess) { cudaGetLastError(); return false; }
        d.raised = true;
    }
    d.pinned++;
    return true;
}
void pin_release(manta_sim *s)   // device current; the simulation's stream already synchronised
{
    std::lock_guard<std::mutex> lock(g_pin_mu);
    PinDevice &d = g_pin[s->device];
    if (d.pinned > 0 && --d.pinned == 0) {
        cudaCtxResetPersistingL2Cache();
        if (d.raised) cudaDeviceSetLimit(cudaLimitPersistingL2CacheSize, d.original);
        cudaGetLastError();
        d.raised = false;
    }
}
void pin_update(manta_sim *s)
{
    const bool want = s->l2_want != 0 && s->live_slots >= MANTA_PIN_MIN_SLOTS;
    if (want && !s->l2_persist) {
        if (pin_acquire(s)) s->l2_persist = s->l2_want;
    } else if (!want && s->l2_persist) {
        cudaStreamSynchronize(s->stream);
        pin_release(s);
        s->l2_persist = 0;
    }
}

// Launch attributes of the step kernels: L2 access-policy window over the occupancy planes (+ cooperative).
int step_attrs(const manta_sim *s, cudaLaunchAttribute *at, bool coop)
{
    int n = 0;
    if (s->l2_persist) {
        at[n].id = cudaLaunchAttributeAccessPolicyWindow;
        at[n].val.accessPolicyWindow.base_ptr = s->l2_window_base;
        at[n].val.accessPolicyWindow.num_bytes = (size_t)s->l2_window_bytes;
        at[n].val.accessPolicyWindow.hitRatio = (float)std::min(1.0, (double)s->l2_persist / (double)s->l2_window_bytes);
        at[n].val.accessPolicyWindow.hitProp = cudaAccessPropertyPersisting;
        at[n].val.accessPolicyWindow.missProp = cudaAccessPropertyStreaming;
        n++;
    }
    if (coop) {
        at[n].id = cudaLaunchAttributeCooperative;
        at[n].val.cooperative = 1;
        n++;
    }
    return n;
}
extern "C++" template <class... KArgs, class... Args>
cudaError_t launch_ks(const manta_sim *s, void (*kern)(KArgs...), int grid, int block, bool coop, size_t smem, Args... args);
extern "C++" template <class... KArgs, class... Args>
cudaError_t launch_k(const manta_sim *s, void (*kern)(KArgs...), int grid, int block, bool coop, Args... args)
{
    return launch_ks(s, kern, grid, block, coop, (size_t)0, args...);
}
extern "C++" template <class... KArgs, class... Args>
cudaError_t launch_ks(const manta_sim *s, void (*kern)(KArgs...), int grid, int block, bool coop, size_t smem, Args... args)
{
    cudaLaunchAttribute at[2];
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)grid);
    cfg.blockDim = dim3((unsigned)block);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = s->stream;
    cfg.attrs = at;
    cfg.numAttrs = (unsigned)step_attrs(s, at, coop);
    return cudaLaunchKernelEx(&cfg, kern, args...);
}

void launch_sort(manta_sim *s, uint32_t t)   // spatial re-sort of the vehicle slots before step t (five stages)
{
    const int from = (int)(((t - 1u) / MANTA_SORT_EVERY) & 1u);
    launch_k(s, k_sort_zero, s->grid_step, MANTA_NT, false, s->P);
    launch_k(s, k_sort_count, s->grid_step, MANTA_NT, false, s->P, from);
    launch_k(s, k_sort_partial, s->grid_step, MANTA_NT, false, s->P);
    launch_k(s, k_sort_scan, s->grid_step, MANTA_NT, false, s->P);
    launch_k(s, k_sort_scatter, s->grid_step, MANTA_NT, false, s->P, from);
    s->launches += 5;
}
bool sort_due_host(uint32_t t) { return t != 0u && t % MANTA_SORT_EVERY == 0u; }

// Kernel-per-phase stepping (MANTA_FLAG_MULTI_KERNEL, manta_step_timed, devices without cooperative launch):
// step t of a call whose last step is t_last.  The admission of step t + 1 rides in the second-phase launch of
// step t when fused; the first step of a call always admits on its own.
void launch_step_multi(manta_sim *s, uint32_t t, bool first, bool last, cudaEvent_t *ev)
{
    if (ev) cudaEventRecord(ev[0], s->stream);
    if (first) {
        if (sort_due_host(t)) launch_sort(s, t);
        launch_k(s, k_admit, s->grid_admit, 256, false, s->P, t);
        s->launches += 1;
    }
    if (ev) cudaEventRecord(ev[1], s->stream);
    launch_ks(s, s->w256 ? k_update<true> : k_update<false>, s->grid_step, MANTA_NT, false, (size_t)MANTA_REC_BYTES, s->P, t);
    if (ev) cudaEventRecord(ev[2], s->stream);
    const int admit_next = (!last && s->fuse_admit) ? 1 : 0;
    launch_k(s, s->w256 ? k_second<true> : k_second<false>, s->grid_step, MANTA_NT, false, s->P, t, admit_next);
    s->launches += 2;
    if (!last) {
        if (sort_due_host(t + 1u)) launch_sort(s, t + 1u);
        if (!admit_next) {
            launch_k(s, k_admit, s->grid_admit, 256, false, s->P, t + 1u);
            s->launches += 1;
        }
    }
    if (ev) cudaEventRecord(ev[3], s->stream);
}

}  // namespace

int manta_step_async(manta_sim *s, uint32_t n_steps)
{
    int rc = check_ready(s, n_steps);
    if (rc) return rc;
    CUDA_TRY(s, cudaSetDevice(s->device));
    pin_update(s);
    if ((s->prm.flags & MANTA_FLAG_MULTI_KERNEL) || s->grid_persist == 0) {
        for (uint32_t k = 0; k < n_steps; k++, s->t++) launch_step_multi(s, s->t, k == 0, k + 1 == n_steps, nullptr);
    } else {
        // one cooperative launch per chunk of timesteps; the grid barrier words restart from zero every launch
        for (uint32_t done = 0; done < n_steps;) {
            uint32_t m = std::min<uint32_t>(n_steps - done, 8192u), t0 = s->t;
            CUDA_TRY(s, cudaMemsetAsync(&s->P.ctr->bar_count, 0, 33 * sizeof(unsigned int), s->stream));   // bar_count .. bar_gen
            CUDA_TRY(s, launch_ks(s, s->w256 ? k_persistent<true> : k_persistent<false>, s->grid_persist, MANTA_NT, true, (size_t)MANTA_REC_BYTES, s->P, t0, m, s->fuse_admit ? 1 : 0));
            s->launches += 1;
            s->t += m;
            done += m;
        }
    }
    CUDA_TRY(s, cudaGetLastError());
    return MANTA_OK;
}

namespace {
extern "C++" template <int NB>
int launch_batch(manta_sim **sims, uint32_t n_sims, uint32_t n_steps, bool w256, int fuse)
{
    manta_sim *s0 = sims[0];
    BatchP<NB> bp{};
    for (uint32_t r = 0; r < (uint32_t)NB; r++) bp.p[r] = sims[std::min(r, n_sims - 1u)]->P;
    void (*kern)(BatchP<NB>, int, uint32_t, uint32_t, int) = w256 ? k_persistent_batch<true, NB> : k_persistent_batch<false, NB>;
    const size_t smem = MANTA_BATCH_SMEM(NB);
    CUDA_TRY(s0, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    int occ = 0;
    CUDA_TRY(s0, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, MANTA_NT, smem));
    if (occ * s0->sm_count < s0->grid_persist)
        return fail(s0, MANTA_ERR_STATE, "a batch of %u simulations does not fit the device next to each other (%d blocks per SM)", n_sims, occ);
    for (uint32_t done = 0; done < n_steps;) {
        const uint32_t m = std::min<uint32_t>(n_steps - done, 8192u), t0 = s0->t + done;
        CUDA_TRY(s0, cudaMemsetAsync(&s0->P.ctr->bar_count, 0, 33 * sizeof(unsigned int), s0->stream));
        cudaLaunchAttribute at[1];
        at[0].id = cudaLaunchAttributeCooperative;
        at[0].val.cooperative = 1;
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3((unsigned)s0->grid_persist);
        cfg.blockDim = dim3(MANTA_NT);
        cfg.dynamicSmemBytes = smem;
        cfg.stream = s0->stream;
        cfg.attrs = at;
        cfg.numAttrs = 1;   // no L2 window: each replica has its own occupancy planes, together beyond the carve-out
        CUDA_TRY(s0, cudaLaunchKernelEx(&cfg, kern, bp, (int)n_sims, t0, m, fuse));
        s0->launches += 1;
        done += m;
    }
    return MANTA_OK;
}
}  // namespace

int manta_step_batch(manta_sim **sims, uint32_t n_sims, uint32_t n_steps)
{
    if (!sims || n_sims == 0 || !sims[0]) return fail(nullptr, MANTA_ERR_INVALID_ARG, "null batch");
    if (n_sims == 1) return manta_step(sims[0], n_steps);
    manta_sim *s0 = sims[0];
    if (n_sims > 4) return fail(s0, MANTA_ERR_INVALID_ARG, "at most 4 simulations per batch");
    bool fuse = true;
    for (uint32_t r = 0; r < n_sims; r++) {
        manta_sim *s = sims[r];
        const int rc = check_ready(s, n_steps);
        if (rc) return rc;
        for (uint32_t q = 0; q < r; q++)
            if (sims[q] == s) return fail(s0, MANTA_ERR_INVALID_ARG, "a simulation appears twice in the batch");
        if (s->device != s0->device || s->stream != s0->stream || s->t != s0->t || s->grid_persist != s0->grid_persist ||
            s->w256 != s0->w256 || s->P.n_seg != s0->P.n_seg || s->grid_persist == 0)
            return fail(s0, MANTA_ERR_INVALID_ARG, "simulations of a batch must share device, stream, step counter and launch geometry "
                                                   "(same look-ahead class, persistent kernel available)");
        fuse = fuse && s->fuse_admit;
    }
    CUDA_TRY(s0, cudaSetDevice(s0->device));
    // A failure once kernels may have run (CUDA error, barrier time-out) leaves EVERY replica mid-step: all of them are
    // marked unusable with the error text, not only the one the error was recorded on.  t advances only after success.
    auto all_unusable = [&](int rc, const manta_sim *src) {
        const std::string msg = "manta_step_batch failed, every simulation of the batch is unusable: " + src->err;
        for (uint32_t r = 0; r < n_sims; r++) {
            sims[r]->sticky_cuda = true;
            sims[r]->err = msg;
        }
        g_last_error = msg;
        return rc;
    };
    int rc = n_sims == 2 ? launch_batch<2>(sims, n_sims, n_steps, s0->w256, fuse ? 1 : 0)
                         : launch_batch<4>(sims, n_sims, n_steps, s0->w256, fuse ? 1 : 0);
    if (rc) return s0->sticky_cuda ? all_unusable(rc, s0) : rc;   // (not sticky: refused before anything was launched)
    if (cudaGetLastError() != cudaSuccess) {
        fail(s0, MANTA_ERR_CUDA, "kernel launch of the batch failed");
        return all_unusable(MANTA_ERR_CUDA, s0);
    }
    for (uint32_t r = 0; r < n_sims; r++) {   // replica 0 first: the barrier words, and with them the abort flag, are its own
        rc = manta_sync(sims[r]);
        if (rc) return all_unusable(rc, sims[r]);
    }
    for (uint32_t r = 0; r < n_sims; r++) sims[r]->t += n_steps;
    return MANTA_OK;
}

int manta_step_timed(manta_sim *s, uint32_t n_steps, double phase_ms[3])
{
    if (!phase_ms) return fail(s, MANTA_ERR_INVALID_ARG, "null argument");
    int rc = check_ready(s, n_steps);
    if (rc) return rc;
    CUDA_TRY(s, cudaSetDevice(s->device));
    pin_update(s);
    const uint32_t CH = 128;
    struct Events {   // destroyed on every return path
        std::vector<cudaEvent_t> ev;
        ~Events() { for (auto e : ev) cudaEventDestroy(e); }
    } E;
    for (uint32_t k = 0; k < 4 * CH; k++) {
        cudaEvent_t e;
        CUDA_TRY(s, cudaEventCreate(&e));
        E.ev.push_back(e);
    }
    std::vector<cudaEvent_t> &ev = E.ev;
    for (uint32_t done = 0; done < n_steps;) {
        const uint32_t m = std::min(CH, n_steps - done);
        for (uint32_t k = 0; k < m; k++, s->t++) launch_step_multi(s, s->t, done + k == 0, done + k + 1 == n_steps, &ev[4 * k]);
        CUDA_TRY(s, cudaStreamSynchronize(s->stream));
        for (uint32_t k = 0; k < m; k++)
            for (int ph = 0; ph < 3; ph++) {
                float ms = 0.f;
                CUDA_TRY(s, cudaEventElapsedTime(&ms, ev[4 * k + ph], ev[4 * k + ph + 1]));
                phase_ms[ph] += (double)ms;
            }
        done += m;
    }
    return MANTA_OK;
}

#ifdef MANTA_DBG
int manta_debug_read(manta_sim *s, uint64_t *out, uint32_t n_words)
{
    cudaStreamSynchronize(s->stream);
    const uint32_t n = std::min<uint32_t>(n_words, s->P.n_seg * 8u);
    cudaMemcpy(out, s->P.dbg_buf, (size_t)n * 8, cudaMemcpyDeviceToHost);
    return (int)s->P.n_seg;
}
#endif

int manta_sync(manta_sim *s)
{
    if (!s) return fail(nullptr, MANTA_ERR_INVALID_ARG, "null simulation");
    CUDA_TRY(s, cudaSetDevice(s->device));
    // both reads are ordered on the stream behind the steps: one synchronisation for the call
    unsigned int ab = 0;
    const bool want_abort = s->loaded && s->grid_persist, want_slots = s->loaded && s->l2_want;
    if (want_abort) CUDA_TRY(s, cudaMemcpyAsync(&ab, &s->P.ctr->abort, sizeof ab, cudaMemcpyDeviceToHost, s->stream));
    if (want_slots) {   // slots in use now (dead ones included): what pin_update goes by
        s->seg_cnt_host.resize(s->P.n_seg);
        CUDA_TRY(s, cudaMemcpyAsync(s->seg_cnt_host.data(), s->P.seg_cnt, (uint64_t)s->P.n_seg * 4, cudaMemcpyDeviceToHost, s->stream));
    }
    CUDA_TRY(s, cudaStreamSynchronize(s->stream));
    if (ab) {
        s->sticky_cuda = true;
        return fail(s, MANTA_ERR_CUDA, "grid barrier of the persistent step kernel timed out");
    }
    if (want_slots) s->live_slots = std::accumulate(s->seg_cnt_host.begin(), s->seg_cnt_host.end(), (uint64_t)0);
    return MANTA_OK;
}

int manta_step(manta_sim *s, uint32_t n_steps)
{
    const int rc = manta_step_async(s, n_steps);
    if (rc) return rc;
    return manta_sync(s);
}

int manta_readback(manta_sim *s, manta_state *st, uint32_t *edge_entries, manta_trip_result *trips, manta_summary *sum)
{
    if (!s) return fail(nullptr, MANTA_ERR_INVALID_ARG, "null simulation");
    if (s->sticky_cuda) return fail(s, MANTA_ERR_CUDA, "earlier CUDA failure");
    if (!s->loaded) return fail(s, MANTA_ERR_STATE, "no trips loaded");
    CUDA_TRY(s, cudaSetDevice(s->device));
    const uint32_t n = s->n_trips;
    if (edge_entries)
        CUDA_TRY(s, cudaMemcpyAsync(edge_entries, s->P.edge_entries, (uint64_t)s->n_edges * 4, cudaMemcpyDeviceToHost, s->stream));
    if (st || trips || sum) {
        // scratch: results uint2 | route_pos u32 | x u32 | v f32 | acc f32 | status u8 | lane u8 | tag u8 | wait u8 | stopped u64
        const uint64_t nn = ((uint64_t)n + 15) & ~15ull;
        const uint64_t scratch = nn * (4 + 16 + 8) + 16;
        uint8_t *buf = (uint8_t *)dev_alloc(s, scratch);
        if (!buf) return fail(s, MANTA_ERR_OOM, "readback scratch allocation failed");
        uint2 *d_res = (uint2 *)buf;
        uint32_t *d_rpos = (uint32_t *)(buf + nn * 8), *d_x = d_rpos + nn;
        float *d_v = (float *)(d_x + nn), *d_acc = d_v + nn;
        uint8_t *d_status = (uint8_t *)(d_acc + nn), *d_lane = d_status + nn, *d_tag = d_lane + nn, *d_wait = d_tag + nn;
        unsigned long long *d_stopped = (unsigned long long *)(d_wait + nn);
        CUDA_TRY(s, cudaMemsetAsync(buf, 0, scratch, s->stream));
        const int g = (int)std::min<uint32_t>((n + 255) / 256, 4096);
        k_status_from_steps<<<g, 256, 0, s->stream>>>(n, s->d_trip_of_id, s->P.admit_step, s->P.arrive_step, d_status, d_res);
        k_gather_state<<<(unsigned)std::min<uint32_t>(s->P.n_seg, 4096u), 256, 0, s->stream>>>(s->P, s->t == 0 ? 0 : (int)(((s->t - 1u) / MANTA_SORT_EVERY) & 1u), s->d_trip_of_id, d_status, d_rpos, d_lane, d_tag, d_x, d_v, d_acc, d_wait, d_stopped);
        CUDA_TRY(s, cudaGetLastError());
        std::vector<uint8_t> h_status(n);
        CUDA_TRY(s, cudaMemcpyAsync(h_status.data(), d_status, n, cudaMemcpyDeviceToHost, s->stream));
        if (st) {
            if (st->route_pos) CUDA_TRY(s, cudaMemcpyAsync(st->route_pos, d_rpos, (uint64_t)n * 4, cudaMemcpyDeviceToHost, s->stream));
            if (st->lane) CUDA_TRY(s, cudaMemcpyAsync(st->lane, d_lane, n, cudaMemcpyDeviceToHost, s->stream));
            if (st->tag) CUDA_TRY(s, cudaMemcpyAsync(st->tag, d_tag, n, cudaMemcpyDeviceToHost, s->stream));
            if (st->x_fx) CUDA_TRY(s, cudaMemcpyAsync(st->x_fx, d_x, (uint64_t)n * 4, cudaMemcpyDeviceToHost, s->stream));
            if (st->v) CUDA_TRY(s, cudaMemcpyAsync(st->v, d_v, (uint64_t)n * 4, cudaMemcpyDeviceToHost, s->stream));
            if (st->acc) CUDA_TRY(s, cudaMemcpyAsync(st->acc, d_acc, (uint64_t)n * 4, cudaMemcpyDeviceToHost, s->stream));
            if (st->wait) CUDA_TRY(s, cudaMemcpyAsync(st->wait, d_wait, n, cudaMemcpyDeviceToHost, s->stream));
        }
        unsigned long long h_stopped = 0;
        CUDA_TRY(s, cudaMemcpyAsync(&h_stopped, d_stopped, sizeof h_stopped, cudaMemcpyDeviceToHost, s->stream));
        if (trips) CUDA_TRY(s, cudaMemcpyAsync(trips, d_res, (uint64_t)n * 8, cudaMemcpyDeviceToHost, s->stream));
        CUDA_TRY(s, cudaStreamSynchronize(s->stream));
        dev_free(s, buf);
        if (st && st->status) memcpy(st->status, h_status.data(), n);
        if (sum) {
            std::vector<BlockStats> bs(s->n_blk_stats);
            CUDA_TRY(s, cudaMemcpy(bs.data(), s->P.blk, sizeof(BlockStats) * bs.size(), cudaMemcpyDeviceToHost));
            memset(sum, 0, sizeof *sum);
            for (uint32_t i = 0; i < n; i++) {
                sum->n_waiting += h_status[i] == MANTA_WAITING;
                sum->n_active += h_status[i] == MANTA_ACTIVE;
            }
            sum->t = s->t;
            sum->n_stopped = h_stopped;
            for (const BlockStats &b : bs) {
                sum->lane_changes += b.lane_changes;
                sum->cells_examined += b.cells_examined;
                sum->lc_evals += b.lc_evals;
                sum->n_done += b.n_done;
                sum->sum_travel_steps += b.sum_travel;
                sum->vehicle_updates += b.n_updates;
            }
        }
    }
    CUDA_TRY(s, cudaStreamSynchronize(s->stream));
    return MANTA_OK;
}

int manta_load_state(manta_sim *s, uint32_t t, const manta_state *st, const manta_trip_result *trips, const uint32_t *edge_entries)
{
    if (!s) return fail(nullptr, MANTA_ERR_INVALID_ARG, "null simulation");
    if (s->sticky_cuda) return fail(s, MANTA_ERR_CUDA, "earlier CUDA failure");
    if (!s->loaded) return fail(s, MANTA_ERR_STATE, "no trips loaded");
    if (!st || !trips || !st->status || !st->route_pos || !st->lane || !st->tag || !st->x_fx || !st->v || t >= 0xFFFFFFF0u)
        return fail(s, MANTA_ERR_INVALID_ARG, "manta_load_state needs status, route_pos, lane, tag, x_fx, v and the trip results");
    CUDA_TRY(s, cudaSetDevice(s->device));
    const uint32_t n = s->n_trips;
    const uint64_t nn = ((uint64_t)n + 15) & ~15ull;
    // scratch: steps uint2 | route_pos u32 | x u32 | v f32 | status u8 | lane u8 | tag u8 | wait u8 | counter, error
    uint8_t *buf = (uint8_t *)dev_alloc(s, nn * (8 + 12 + 4) + 16);
    if (!buf) return fail(s, MANTA_ERR_OOM, "state scratch allocation failed");
    uint2 *d_steps = (uint2 *)buf;
    uint32_t *d_rpos = (uint32_t *)(buf + nn * 8), *d_x = d_rpos + nn;
    float *d_v = (float *)(d_x + nn);
    uint8_t *d_status = (uint8_t *)(d_v + nn), *d_lane = d_status + nn, *d_tag = d_lane + nn, *d_wait = d_tag + nn;
    uint32_t *d_counter = (uint32_t *)(d_wait + nn), *d_err = d_counter + 1;
    auto done = [&](int rc) { cudaStreamSynchronize(s->stream); dev_free(s, buf); return rc; };
#define TRY_LS(expr) do { cudaError_t e_ = (expr); if (e_ != cudaSuccess) { s->sticky_cuda = true; return done(fail(s, MANTA_ERR_CUDA, "%s: %s", #expr, cudaGetErrorString(e_))); } } while (0)
    TRY_LS(cudaMemsetAsync(d_counter, 0, 8, s->stream));
    TRY_LS(cudaMemcpyAsync(d_steps, trips, (uint64_t)n * 8, cudaMemcpyHostToDevice, s->stream));
    TRY_LS(cudaMemcpyAsync(d_rpos, st->route_pos, (uint64_t)n * 4, cudaMemcpyHostToDevice, s->stream));
    TRY_LS(cudaMemcpyAsync(d_x, st->x_fx, (uint64_t)n * 4, cudaMemcpyHostToDevice, s->stream));
    TRY_LS(cudaMemcpyAsync(d_v, st->v, (uint64_t)n * 4, cudaMemcpyHostToDevice, s->stream));
    TRY_LS(cudaMemcpyAsync(d_status, st->status, n, cudaMemcpyHostToDevice, s->stream));
    TRY_LS(cudaMemcpyAsync(d_lane, st->lane, n, cudaMemcpyHostToDevice, s->stream));
    TRY_LS(cudaMemcpyAsync(d_tag, st->tag, n, cudaMemcpyHostToDevice, s->stream));
    if (st->wait) TRY_LS(cudaMemcpyAsync(d_wait, st->wait, n, cudaMemcpyHostToDevice, s->stream));
    StateIn in{d_status, d_lane, d_tag, st->wait ? d_wait : nullptr, d_rpos, d_x, d_v, d_steps};
    const int g = (int)std::min<uint32_t>((std::max(n, s->P.n_queues) + 255) / 256, 4096);
    // pass 1: validation only -- a bad state leaves the simulation as it was
    k_state_validate<<<g, 256, 0, s->stream>>>(s->P, in, s->d_trip_of_id, n, t, d_err);
    uint32_t h_err = 0;
    TRY_LS(cudaMemcpyAsync(&h_err, d_err, 4, cudaMemcpyDeviceToHost, s->stream));
    TRY_LS(cudaStreamSynchronize(s->stream));
    if (h_err) {
        static const char *what[] = {"", "status value above 2", "route position beyond the trip's route",
                                     "lane, position or stop counter out of range, or a speed that is negative, not finite or above the fastest possible one (largest desired or initial speed + a dt)",
                                     "an admitted trip stands behind a waiting one of the same origin edge (admission is first in, first out)",
                                     "admit / arrive steps that contradict the status (WAITING: none; ACTIVE: admit_step <= t, no arrive_step; DONE: admit_step <= arrive_step <= t)"};
        return done(fail(s, MANTA_ERR_INVALID_ARG, "manta_load_state: %s", what[std::min<uint32_t>(h_err, 5u)]));
    }
    // pass 2: rebuild.  Both occupancy planes empty (no vehicle has an earlier mark), claims unclaimed, counters restarted.
    const uint64_t plane_words = ((s->n_cells / 64 + 8) + 15) & ~15ull;
    TRY_LS(cudaMemsetAsync(s->P.bits[0], 0, 2 * plane_words * sizeof(u64), s->stream));
    TRY_LS(cudaMemsetAsync(s->P.claim, 0xFF, ((uint64_t)s->n_edges * 8 + s->n_nodes) * sizeof(u64), s->stream));
    TRY_LS(cudaMemsetAsync(s->P.blk, 0, sizeof(BlockStats) * s->n_blk_stats, s->stream));
    if (edge_entries) TRY_LS(cudaMemcpyAsync(s->P.edge_entries, edge_entries, (uint64_t)s->n_edges * 4, cudaMemcpyHostToDevice, s->stream));
    const int sb = t == 0 ? 0 : (int)(((t - 1u) / MANTA_SORT_EVERY) & 1u);
    k_state_load<<<g, 256, 0, s->stream>>>(s->P, in, s->d_trip_of_id, n, t, sb, d_counter, d_err);
    k_state_counts<<<(s->P.n_seg + 255) / 256, 256, 0, s->stream>>>(s->P, d_counter);
    s->launches += 3;
    TRY_LS(cudaGetLastError());
    uint32_t h_tail[2] = {0u, 0u};   // {slots dealt out, error}
    TRY_LS(cudaMemcpyAsync(h_tail, d_counter, 8, cudaMemcpyDeviceToHost, s->stream));
    TRY_LS(cudaStreamSynchronize(s->stream));
#undef TRY_LS
    h_err = h_tail[1];
    s->live_slots = h_tail[0];
    s->t = t;
    if (h_err) {   // found while rebuilding: the state is unusable now
        s->sticky_cuda = true;
        return done(fail(s, MANTA_ERR_INVALID_ARG, "manta_load_state: two vehicles in one atlas cell; the simulation must be destroyed"));
    }
    return done(MANTA_OK);
}

int manta_check_failures(manta_sim *s)
{
#ifdef MANTA_CHECK
    if (!s) return -1;
    cudaSetDevice(s->device);
    cudaStreamSynchronize(s->stream);
    CheckCtx c{};
    if (cudaMemcpyFromSymbol(&c, g_check, sizeof c) != cudaSuccess) return -1;
    return (int)c.fail;
#else
    (void)s;
    return -1;
#endif
}

int manta_readback_edge_speeds(manta_sim *s, uint64_t *sum_q8, uint32_t *samples)
{
    if (!s) return fail(nullptr, MANTA_ERR_INVALID_ARG, "null simulation");
    if (s->sticky_cuda) return fail(s, MANTA_ERR_CUDA, "earlier CUDA failure");
    if (!s->P.stat_n_slices) return fail(s, MANTA_ERR_STATE, "per-edge speed statistics are off (manta_params.stat_period_steps = 0)");
    CUDA_TRY(s, cudaSetDevice(s->device));
    const uint64_t n = (uint64_t)s->P.stat_n_slices * s->n_edges;
    if (sum_q8) CUDA_TRY(s, cudaMemcpyAsync(sum_q8, s->P.stat_sum, n * sizeof(uint64_t), cudaMemcpyDeviceToHost, s->stream));
    if (samples) CUDA_TRY(s, cudaMemcpyAsync(samples, s->P.stat_cnt, n * sizeof(uint32_t), cudaMemcpyDeviceToHost, s->stream));
    CUDA_TRY(s, cudaStreamSynchronize(s->stream));
    return MANTA_OK;
}

int manta_readback_atlas(manta_sim *s, uint16_t *occ, float *spd, uint32_t *cell_off, uint32_t *pitch)
{
    if (!s) return fail(nullptr, MANTA_ERR_INVALID_ARG, "null simulation");
    if (s->sticky_cuda) return fail(s, MANTA_ERR_CUDA, "earlier CUDA failure");
    CUDA_TRY(s, cudaSetDevice(s->device));
    if (occ || spd) {
        // the logical atlas is rebuilt from the occupancy bits and the payload plane of the current step
        const uint64_t n = s->n_cells;
        uint8_t *buf = (uint8_t *)dev_alloc(s, n * 6 + 64);
        if (!buf) return fail(s, MANTA_ERR_OOM, "atlas export scratch allocation failed");
        float *d_spd = (float *)buf;
        uint16_t *d_occ = (uint16_t *)(buf + n * 4);
        k_export_atlas<<<(unsigned)std::min<uint64_t>((n + 255) / 256, 65535ull), 256, 0, s->stream>>>(
            s->P.bits[s->t & 1u], s->P.pay[s->t & 1u], s->P.pay_shift, n, d_occ, d_spd);
        CUDA_TRY(s, cudaGetLastError());
        if (occ) CUDA_TRY(s, cudaMemcpyAsync(occ, d_occ, n * 2, cudaMemcpyDeviceToHost, s->stream));
        if (spd) CUDA_TRY(s, cudaMemcpyAsync(spd, d_spd, n * 4, cudaMemcpyDeviceToHost, s->stream));
        CUDA_TRY(s, cudaStreamSynchronize(s->stream));
        dev_free(s, buf);
    }
    for (uint32_t e = 0; e < s->n_edges; e++) {
        if (cell_off) cell_off[e] = s->cell_off[e];
        if (pitch) pitch[e] = (s->len_c[e] + 63u) & ~63u;
    }
    return MANTA_OK;
}


int manta_selftest_grid_barrier(int cuda_device, uint32_t n_rounds, uint64_t *n_stale, uint32_t *n_blocks)
{
    if (!n_stale || n_rounds == 0 || n_rounds > (1u << 22)) return fail(nullptr, MANTA_ERR_INVALID_ARG, "manta_selftest_grid_barrier: null result or 0 / more than 2^22 rounds");
    int n_dev = 0, sms = 0, coop = 0, occ = 0;
    if (cudaGetDeviceCount(&n_dev) != cudaSuccess || cuda_device < 0 || cuda_device >= n_dev) {
        cudaGetLastError();
        return fail(nullptr, MANTA_ERR_CUDA, "no CUDA device %d (there is no CPU fallback)", cuda_device);
    }
    CUDA_TRY((manta_sim *)nullptr, cudaSetDevice(cuda_device));
    CUDA_TRY((manta_sim *)nullptr, cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, cuda_device));
    CUDA_TRY((manta_sim *)nullptr, cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, cuda_device));
    CUDA_TRY((manta_sim *)nullptr, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_barrier_litmus, MANTA_NT, 0));
    if (!coop || occ < 1) return fail(nullptr, MANTA_ERR_STATE, "cooperative launches are not available on device %d", cuda_device);
    const int grid = sms * std::min(occ, MANTA_MINB);   // the persistent step kernel's geometry: MANTA_MINB blocks of MANTA_NT threads per SM
    uint8_t *buf = nullptr;
    const size_t words_off = sizeof(Counters), stale_off = words_off + (size_t)grid * 32 * 4, total = stale_off + 8;
    CUDA_TRY((manta_sim *)nullptr, cudaMalloc(&buf, total));
    int rc = MANTA_OK;
    cudaError_t e = cudaMemset(buf, 0, total);
    if (e == cudaSuccess) {
        Counters *c = (Counters *)buf;
        uint32_t *words = (uint32_t *)(buf + words_off);
        unsigned long long *stale = (unsigned long long *)(buf + stale_off);
        void *args[] = {&c, &words, &n_rounds, &stale};
        e = cudaLaunchCooperativeKernel((const void *)k_barrier_litmus, dim3((unsigned)grid), dim3(MANTA_NT), args, 0, 0);
        if (e == cudaSuccess) e = cudaDeviceSynchronize();
        unsigned long long h_stale = 0;
        unsigned int h_abort = 0, h_count = 0;
        if (e == cudaSuccess) e = cudaMemcpy(&h_stale, stale, 8, cudaMemcpyDeviceToHost);
        if (e == cudaSuccess) e = cudaMemcpy(&h_abort, &c->abort, 4, cudaMemcpyDeviceToHost);
        if (e == cudaSuccess) e = cudaMemcpy(&h_count, &c->bar_count, 4, cudaMemcpyDeviceToHost);
        if (e == cudaSuccess) {
            *n_stale = h_stale;
            if (n_blocks) *n_blocks = (uint32_t)grid;
            if (h_abort) rc = fail(nullptr, MANTA_ERR_CUDA, "grid barrier timed out in the self-test");
#if MANTA_BAR >= 1
            else if (h_count != 2u * n_rounds * (unsigned)grid)   // every block arrived at every barrier
                rc = fail(nullptr, MANTA_ERR_CUDA, "grid barrier self-test: %u arrivals counted, %u expected", h_count, 2u * n_rounds * (unsigned)grid);
#endif
        }
    }
    if (e != cudaSuccess) rc = fail(nullptr, MANTA_ERR_CUDA, "grid barrier self-test: %s", cudaGetErrorString(e));
    cudaFree(buf);
    return rc;
}

// ---- manta_readback_noalloc: manta_readback without any device allocation ------------------------------------------
namespace {
constexpr int kNoallocMaxDevices = 64;
std::mutex g_noalloc_mu;                              // one call at a time per process: every call uses the same array
void *g_noalloc_ptr[kNoallocMaxDevices] = {};         // device address of g_noalloc_scratch, per device ordinal
}  // namespace

int manta_readback_noalloc(manta_sim *s, manta_state *st, uint32_t *edge_entries, manta_trip_result *trips, manta_summary *sum)
{
    if (!s) return fail(nullptr, MANTA_ERR_INVALID_ARG, "null simulation");
    if (s->sticky_cuda) return fail(s, MANTA_ERR_CUDA, "earlier CUDA failure");
    if (!s->loaded) return fail(s, MANTA_ERR_STATE, "no trips loaded");
    const uint32_t n = s->n_trips;
    if (n > MANTA_NOALLOC_MAX_TRIPS)
        return fail(s, MANTA_ERR_INVALID_ARG, "manta_readback_noalloc: %u trips exceed the built-in scratch of MANTA_NOALLOC_MAX_TRIPS = %u trips; use manta_readback",
                    n, MANTA_NOALLOC_MAX_TRIPS);
    if (s->device < 0 || s->device >= kNoallocMaxDevices)
        return fail(s, MANTA_ERR_INVALID_ARG, "manta_readback_noalloc: device ordinal %d beyond the %d this call keeps an address for", s->device, kNoallocMaxDevices);
    CUDA_TRY(s, cudaSetDevice(s->device));
    std::lock_guard<std::mutex> lock(g_noalloc_mu);   // held until the results are on the host: the array is shared
    if (!g_noalloc_ptr[s->device]) {
        // set-up, once per device, with that device current: the array's address on THIS device
        void *p = nullptr;
        CUDA_TRY(s, cudaGetSymbolAddress(&p, g_noalloc_scratch));
        g_noalloc_ptr[s->device] = p;
    }
    uint8_t *buf = (uint8_t *)g_noalloc_ptr[s->device];
    if (edge_entries)
        CUDA_TRY(s, cudaMemcpyAsync(edge_entries, s->P.edge_entries, (uint64_t)s->n_edges * 4, cudaMemcpyDeviceToHost, s->stream));
    if (st || trips || sum) {
        // same staging layout as manta_readback, inside the static array
        const uint64_t nn = ((uint64_t)n + 15) & ~15ull;
        const uint64_t used = nn * MANTA_NOALLOC_BYTES_PER_TRIP + 16;
        uint2 *d_res = (uint2 *)buf;
        uint32_t *d_rpos = (uint32_t *)(buf + nn * 8), *d_x = d_rpos + nn;
        float *d_v = (float *)(d_x + nn), *d_acc = d_v + nn;
        uint8_t *d_status = (uint8_t *)(d_acc + nn), *d_lane = d_status + nn, *d_tag = d_lane + nn, *d_wait = d_tag + nn;
        unsigned long long *d_stopped = (unsigned long long *)(d_wait + nn);
        // the array still holds the previous call's rows and stop count: everything read below starts from zero
        CUDA_TRY(s, cudaMemsetAsync(buf, 0, used, s->stream));
        const int g = (int)std::min<uint32_t>((n + 255) / 256, 4096);
        k_status_from_steps<<<g, 256, 0, s->stream>>>(n, s->d_trip_of_id, s->P.admit_step, s->P.arrive_step, d_status, d_res);
        k_gather_state<<<(unsigned)std::min<uint32_t>(s->P.n_seg, 4096u), 256, 0, s->stream>>>(s->P, s->t == 0 ? 0 : (int)(((s->t - 1u) / MANTA_SORT_EVERY) & 1u), s->d_trip_of_id, d_status, d_rpos, d_lane, d_tag, d_x, d_v, d_acc, d_wait, d_stopped);
        CUDA_TRY(s, cudaGetLastError());
        std::vector<uint8_t> own_status;   // host memory only, and only when the caller gave no status array
        uint8_t *h_status = st && st->status ? st->status : nullptr;
        if (!h_status && sum) {
            own_status.resize(n);
            h_status = own_status.data();
        }
        if (h_status) CUDA_TRY(s, cudaMemcpyAsync(h_status, d_status, n, cudaMemcpyDeviceToHost, s->stream));
        if (st) {
            if (st->route_pos) CUDA_TRY(s, cudaMemcpyAsync(st->route_pos, d_rpos, (uint64_t)n * 4, cudaMemcpyDeviceToHost, s->stream));
            if (st->lane) CUDA_TRY(s, cudaMemcpyAsync(st->lane, d_lane, n, cudaMemcpyDeviceToHost, s->stream));
            if (st->tag) CUDA_TRY(s, cudaMemcpyAsync(st->tag, d_tag, n, cudaMemcpyDeviceToHost, s->stream));
            if (st->x_fx) CUDA_TRY(s, cudaMemcpyAsync(st->x_fx, d_x, (uint64_t)n * 4, cudaMemcpyDeviceToHost, s->stream));
            if (st->v) CUDA_TRY(s, cudaMemcpyAsync(st->v, d_v, (uint64_t)n * 4, cudaMemcpyDeviceToHost, s->stream));
            if (st->acc) CUDA_TRY(s, cudaMemcpyAsync(st->acc, d_acc, (uint64_t)n * 4, cudaMemcpyDeviceToHost, s->stream));
            if (st->wait) CUDA_TRY(s, cudaMemcpyAsync(st->wait, d_wait, n, cudaMemcpyDeviceToHost, s->stream));
        }
        unsigned long long h_stopped = 0;
        CUDA_TRY(s, cudaMemcpyAsync(&h_stopped, d_stopped, sizeof h_stopped, cudaMemcpyDeviceToHost, s->stream));
        if (trips) CUDA_TRY(s, cudaMemcpyAsync(trips, d_res, (uint64_t)n * 8, cudaMemcpyDeviceToHost, s->stream));
        CUDA_TRY(s, cudaStreamSynchronize(s->stream));
        if (sum) {
            std::vector<BlockStats> bs(s->n_blk_stats);
            CUDA_TRY(s, cudaMemcpy(bs.data(), s->P.blk, sizeof(BlockStats) * bs.size(), cudaMemcpyDeviceToHost));
            memset(sum, 0, sizeof *sum);
            for (uint32_t i = 0; i < n; i++) {
                sum->n_waiting += h_status[i] == MANTA_WAITING;
                sum->n_active += h_status[i] == MANTA_ACTIVE;
            }
            sum->t = s->t;
            sum->n_stopped = h_stopped;
            for (const BlockStats &b : bs) {
                sum->lane_changes += b.lane_changes;
                sum->cells_examined += b.cells_examined;
                sum->lc_evals += b.lc_evals;
                sum->n_done += b.n_done;
                sum->sum_travel_steps += b.sum_travel;
                sum->vehicle_updates += b.n_updates;
            }
        }
    }
    CUDA_TRY(s, cudaStreamSynchronize(s->stream));
    return MANTA_OK;
}

}  // extern "C"

// libsw.so -- C ABI of include/sw.h: context, host-side scheduling of the sweep kernels, copies.
// All arithmetic of the method runs in the kernels of sw_generic.cuh / sw_tile.cuh; the only host
// arithmetic is the threshold table (double precision, once per context; R6/R7).
#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <utility>
#include <vector>

#include "sw.h"
#include "sw_generic.cuh"
#include "sw_paper_ccl.cuh"
#include "sw_philox.cuh"
#include "sw_small.cuh"
#include "sw_tile.cuh"

namespace {

thread_local char g_err[512] = "";

int fail(int code, const char *fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
    return code;
}

#define CU_TRY(expr)                                                                              \
    do {                                                                                          \
        cudaError_t e_ = (expr);                                                                  \
        if (e_ != cudaSuccess)                                                                    \
            return fail(e_ == cudaErrorMemoryAllocation ? SW_ERR_NOMEM : SW_ERR_CUDA, "%s: %s",   \
                        #expr, cudaGetErrorString(e_));                                           \
    } while (0)

constexpr size_t ALIGN = 1024;
constexpr int REC_ROWS = 512;  // rows of the device ring used by sw_sweep_record
constexpr int OBS_WORDS = 64;  // [0,16) bond_hist, [16,32) state_hist, [32,48) corr_hist(r1), [48,64) corr_hist(r2)

size_t align_up(size_t x) { return (x + ALIGN - 1) / ALIGN * ALIGN; }

bool args_ok(int L, int q, int model)
{
    return L >= 2 && L <= SW_MAX_L && q >= 2 && q <= SW_MAX_Q && (model == SW_POTTS || model == SW_CLOCK);
}

struct Carve {
    size_t spins, spins2, labels, labels2, bonds, table, obs, flag, stats, ring, small, tiled, total;
};

Carve carve(int L, int q)
{
    (void)q;
    const size_t N = (size_t)L * (size_t)L;
    Carve c;
    size_t off = 0;
    c.spins = off;  off += align_up(N);
    c.spins2 = off; off += align_up(N);
    c.labels = off; off += align_up(4 * N);
    c.labels2 = off; off += align_up(4 * N);     // R of the Hawick labeller (SW_ALGO_HAWICK)
    c.bonds = off;  off += align_up(N);
    c.table = off;  off += align_up(4 * (size_t)(2 * SW_MAX_Q) * (2 * SW_MAX_Q));
    c.obs = off;    off += align_up(8 * OBS_WORDS);
    c.flag = off;   off += align_up(64);
    c.stats = off;  off += align_up(8 * SW_NUM_STATS);
    c.ring = off;   off += align_up((size_t)REC_ROWS * OBS_WORDS * 8);
    c.small = off;  off += align_up(sizeof(sw::SmallLattice));
    c.tiled = off;  off += align_up(sw::tiled_workspace_bytes(L));
    c.total = off;
    return c;
}

}  // namespace

struct sw_ctx {
    int L = 0, q = 0, model = 0;
    double T = 0.0;
    uint64_t seed = 0, t = 0;
    size_t N = 0;
    cudaStream_t stream = nullptr;
    int device = 0, sms = 148;      // the device the workspace and stream belong to; its SM count (grid sizing)
    bool own_stream = false, own_ws = false;
    char *ws = nullptr;
    Carve cv{};
    uint8_t *spins = nullptr, *spins_alt = nullptr, *bonds = nullptr;  // spins = S^t; spins_alt = the other buffer of the tiled ping-pong
    int32_t *labels = nullptr, *labels2 = nullptr;
    uint32_t *table = nullptr;
    unsigned long long *obs = nullptr, *stats = nullptr, *ring = nullptr;
    int *flag = nullptr;
    char *tiled_ws = nullptr;
    sw::SmallLattice *small_lat = nullptr;   // device: key and threshold of this lattice, as the one-CTA kernel reads them
    sw::Model md{};
    sw::PhiloxKey key{};
    std::vector<uint32_t> thr_host;  // 1 (Potts) or (2q)^2 (clock)
    int algo = SW_ALGO_GENERIC;
    bool have_labels = false, stats_on = false;
    int last_algo = 0;
    uint64_t launches = 0, stat_sweeps = 0;
    uint64_t ccl_iterations = 0, ccl_sweeps = 0;   // SW_ALGO_HAWICK / SW_ALGO_KALENTEV: scan passes and the sweeps they served
    sw::TiledState tiled{};
    unsigned long long *rec_host = nullptr;   // pinned copy of the record ring (sw_sweep_record)
    // Tiled back-end: chunks of GRAPH_SWEEPS sweeps replayed from a CUDA graph (one per parity of the spin ping-pong).
    // The sweep index stays a kernel parameter (a uniform value the compiler keeps in uniform registers): before a
    // replay the t of the 2 * GRAPH_SWEEPS kernel nodes that take one is set with cudaGraphExecKernelNodeSetParams.
    struct GraphNode {
        cudaGraphNode_t node;
        cudaKernelNodeParams params;      // as captured; kernelParams replaced by `kp`
        std::vector<void *> kp;           // the node's parameter pointers, entry 2 (t) redirected to `t`
        uint32_t offset, t;               // sweep inside the chunk; value for the next replay
    };
    struct SweepGraph {
        cudaGraph_t graph = nullptr;      // kept alive: the captured parameter storage belongs to it
        cudaGraphExec_t exec = nullptr;
        std::vector<GraphNode> nodes;
    } graph[2];
    uint64_t graph_replays = 0;
    bool graph_off = false;                   // SW_NO_GRAPH=1, or capture failed once: plain launches from then on
};

namespace {

// A context belongs to the device that was current when it was created: every entry point makes that device current
// for its own duration and restores the caller's on return.
struct DeviceGuard {
    int prev = -1;
    bool switched = false;
    explicit DeviceGuard(const sw_ctx *c)
    {
        if (c && cudaGetDevice(&prev) == cudaSuccess && prev != c->device) switched = cudaSetDevice(c->device) == cudaSuccess;
    }
    ~DeviceGuard() { if (switched) cudaSetDevice(prev); }
};

uint32_t thr_from_p(double p)
{
    double v = std::floor(p * 4294967296.0);
    if (!(v > 0.0)) return 0u;
    if (v >= 4294967295.0) return 0xFFFFFFFFu;
    return (uint32_t)v;
}

// DESIGN.md R1 (Potts) and R4 (clock).  Host, double precision.
void build_thresholds(sw_ctx *c)
{
    if (c->model == SW_POTTS) {
        c->thr_host.assign(1, thr_from_p(1.0 - std::exp(-1.0 / c->T)));
    } else {
        const int n = 2 * c->q;
        const double pi = 3.14159265358979323846;
        c->thr_host.assign((size_t)n * n, 0u);
        std::vector<double> s(n);
        for (int k = 0; k < n; ++k) s[k] = (k % c->q == 0) ? 0.0 : std::sin(pi * (double)k / (double)c->q);
        for (int a = 0; a < n; ++a)
            for (int b = 0; b < n; ++b) {
                const double pr = s[a] * s[b];
                if (pr > 0.0) c->thr_host[(size_t)a * n + b] = thr_from_p(1.0 - std::exp(-2.0 * pr / c->T));
            }
    }
}

inline unsigned blocks_for(size_t n, unsigned bs) { return (unsigned)((n + bs - 1) / bs); }

const char *const GENERIC_KERNELS[] = { "k_bonds", "k_label_init", "k_union", "k_flatten", "k_flip" };

// One sweep with one of the paper's own labellers: bonds -> iterated label equivalence -> flip.
int paper_sweep(sw_ctx *c, uint32_t t, cudaEvent_t *ev)
{
    const unsigned bs = 256;
    const uint32_t N = c->md.N;
    if (ev) cudaEventRecord(ev[0], c->stream);
    sw::k_bonds<<<blocks_for((N + 1) / 2, bs), bs, 0, c->stream>>>(c->md, c->key, t, c->spins, c->bonds);
    if (ev) cudaEventRecord(ev[1], c->stream);
    const int it = sw::paper_ccl_label(c->algo == SW_ALGO_KALENTEV, c->md, c->bonds, c->labels, c->labels2, c->flag, c->stream, &c->launches);
    if (it < 0) return fail(SW_ERR_CUDA, "paper labeller failed: %s", cudaGetErrorString(cudaGetLastError()));
    c->ccl_iterations += (uint64_t)it;
    c->ccl_sweeps += 1;
    if (ev) cudaEventRecord(ev[2], c->stream);
    sw::k_flip<<<blocks_for(N, bs), bs, 0, c->stream>>>(c->md, c->key, t, c->labels, c->spins);
    if (ev) cudaEventRecord(ev[3], c->stream);
    c->launches += 2;
    CU_TRY(cudaPeekAtLastError());
    return SW_OK;
}

// SW_ALGO_AUTO: one CTA for L <= 64 (measured: 7 us per sweep at L = 32 and 26 us at L = 64 against 22 and 28 us of
// the five generic launches; at L = 128 the single CTA is the slower one), tiles when L allows them, else generic
int auto_algo(int L)
{
    return L <= 64 ? SW_ALGO_SMALL : sw::tiled_supported(L) ? SW_ALGO_TILED : SW_ALGO_GENERIC;
}

// n sweeps of the one-CTA back-end in ONE launch (sweep indices c->t .. c->t + n - 1; labels of the last one exported)
int small_sweeps(sw_ctx *c, int n, cudaEvent_t *ev = nullptr)
{
    if (ev) cudaEventRecord(ev[0], c->stream);
    CU_TRY(sw::small_launch(c->model, 1, c->L, c->q, c->small_lat, c->table, c->spins, c->labels, (uint32_t)c->t, n, c->stream,
                             c->stats_on ? c->stats : nullptr));
    if (ev) cudaEventRecord(ev[1], c->stream);
    c->launches += 1;
    return SW_OK;
}

// ev (optional): ev[0] is recorded before the first kernel, ev[k+1] after kernel k.
int generic_sweep(sw_ctx *c, uint32_t t, cudaEvent_t *ev)
{
    const unsigned bs = 256;
    const uint32_t N = c->md.N;
    if (ev) cudaEventRecord(ev[0], c->stream);
    sw::k_bonds<<<blocks_for((N + 1) / 2, bs), bs, 0, c->stream>>>(c->md, c->key, t, c->spins, c->bonds);
    if (ev) cudaEventRecord(ev[1], c->stream);
    sw::k_label_init<<<blocks_for(N, bs), bs, 0, c->stream>>>(N, c->labels);
    if (ev) cudaEventRecord(ev[2], c->stream);
    sw::k_union<<<blocks_for(N, bs), bs, 0, c->stream>>>(c->md, c->bonds, c->labels);
    if (ev) cudaEventRecord(ev[3], c->stream);
    sw::k_flatten<<<blocks_for(N, bs), bs, 0, c->stream>>>(N, c->labels);
    if (ev) cudaEventRecord(ev[4], c->stream);
    sw::k_flip<<<blocks_for(N, bs), bs, 0, c->stream>>>(c->md, c->key, t, c->labels, c->spins);
    if (ev) cudaEventRecord(ev[5], c->stream);
    c->launches += 5;
    CU_TRY(cudaPeekAtLastError());
    return SW_OK;
}

// obs_row (optional): zeroed row of the record ring that receives the observables of S^t if the back-end fuses S5 into
// its first kernel (fuses_observables); otherwise the caller has launched k_observables on it already.
bool fuses_observables(const sw_ctx *c) { return c->algo == SW_ALGO_TILED && !c->stats_on && sw::tiled_fuses_observables(c->md); }

// sw_sweep(n) of the tiled back-end, n >= GRAPH_SWEEPS: the 3 kernels of GRAPH_SWEEPS consecutive sweeps (with their
// programmatic-dependent-launch edges) are captured once per ping-pong parity and replayed with one cudaGraphLaunch per
// chunk, after the sweep indices of its nodes have been set ("CUDA graph or persistent kernel" as the host
// scheduler).  GRAPH_SWEEPS is even, so a chunk leaves the roles of the two spin buffers as it found them.
constexpr int GRAPH_SWEEPS = 16;

bool build_graph(sw_ctx *c, int which)
{
    // captured on a private stream (the context's may be the legacy default stream, which cannot capture); nothing runs
    // on it: the instantiated graph is launched on the context's stream
    sw_ctx::SweepGraph &sg = c->graph[which];
    cudaStream_t cap = nullptr;
    if (cudaStreamCreateWithFlags(&cap, cudaStreamNonBlocking) != cudaSuccess) { cudaGetLastError(); return false; }
    if (cudaStreamBeginCapture(cap, cudaStreamCaptureModeThreadLocal) != cudaSuccess) { cudaGetLastError(); cudaStreamDestroy(cap); return false; }
    uint8_t *a = c->spins, *b = c->spins_alt;
    uint64_t dummy = 0;
    bool ok = true;
    for (int s = 0; s < GRAPH_SWEEPS && ok; ++s) {
        ok = sw::tiled_sweep(c->tiled, c->md, c->key, (uint32_t)s, a, b, (unsigned long long *)c->labels, cap, nullptr, &dummy, nullptr) == 0;
        std::swap(a, b);
    }
    if (cudaStreamEndCapture(cap, &sg.graph) != cudaSuccess || !sg.graph) ok = false;
    cudaStreamDestroy(cap);
    if (ok && cudaGraphInstantiate(&sg.exec, sg.graph, 0) != cudaSuccess) { sg.exec = nullptr; ok = false; }
    // the kernel nodes that take the sweep index (parameter 2 of the labeling and of the flip kernel; captured with t = the
    // sweep's offset inside the chunk, which identifies them)
    size_t n = 0;
    if (ok && cudaGraphGetNodes(sg.graph, nullptr, &n) != cudaSuccess) ok = false;
    std::vector<cudaGraphNode_t> all(n);
    if (ok && n && cudaGraphGetNodes(sg.graph, all.data(), &n) != cudaSuccess) ok = false;
    const void *label_fn = c->model == SW_POTTS ? (const void *)sw::k_tile_label<0, false, false> : (const void *)sw::k_tile_label<1, false, false>;
    const void *flip_fn = c->model == SW_POTTS ? (const void *)sw::k_tile_flip<0, false> : (const void *)sw::k_tile_flip<1, false>;
    for (size_t k = 0; ok && k < n; ++k) {
        cudaGraphNodeType type;
        if (cudaGraphNodeGetType(all[k], &type) != cudaSuccess) { ok = false; break; }
        if (type != cudaGraphNodeTypeKernel) continue;
        sw_ctx::GraphNode gn;
        gn.node = all[k];
        if (cudaGraphKernelNodeGetParams(all[k], &gn.params) != cudaSuccess) { ok = false; break; }
        const int np = gn.params.func == label_fn ? 16 : gn.params.func == flip_fn ? 10 : 0;
        if (np == 0) continue;                        // k_seam_merge takes no sweep index
        gn.kp.assign(gn.params.kernelParams, gn.params.kernelParams + np);
        gn.offset = *static_cast<const uint32_t *>(gn.kp[2]);
        gn.t = gn.offset;
        sg.nodes.push_back(std::move(gn));
    }
    ok = ok && sg.nodes.size() == 2u * GRAPH_SWEEPS;
    if (!ok) {
        if (sg.exec) cudaGraphExecDestroy(sg.exec);
        if (sg.graph) cudaGraphDestroy(sg.graph);
        sg.exec = nullptr; sg.graph = nullptr; sg.nodes.clear();
        cudaGetLastError();
    }
    return ok;
}

// as many whole chunks of n sweeps as possible through the graphs; returns the number of sweeps done (0: none)
int graph_sweeps(sw_ctx *c, int n)
{
    int done = 0;
    while (n - done >= GRAPH_SWEEPS && !c->graph_off) {
        const int which = c->spins == c->tiled.map_base[0] ? 0 : 1;
        sw_ctx::SweepGraph &sg = c->graph[which];
        if (!sg.exec && !build_graph(c, which)) { c->graph_off = true; break; }
        bool ok = true;
        for (sw_ctx::GraphNode &gn : sg.nodes) {
            gn.t = (uint32_t)c->t + gn.offset;
            gn.kp[2] = &gn.t;
            gn.params.kernelParams = gn.kp.data();
            ok = ok && cudaGraphExecKernelNodeSetParams(sg.exec, gn.node, &gn.params) == cudaSuccess;
        }
        if (!ok || cudaGraphLaunch(sg.exec, c->stream) != cudaSuccess) { cudaGetLastError(); c->graph_off = true; break; }
        c->t += GRAPH_SWEEPS;
        c->launches += 3 * GRAPH_SWEEPS;
        c->graph_replays += 1;
        done += GRAPH_SWEEPS;
        c->last_algo = c->algo;
        c->have_labels = true;
    }
    return done;
}

int one_sweep(sw_ctx *c, cudaEvent_t *ev = nullptr, unsigned long long *obs_row = nullptr)
{
    const uint32_t t = (uint32_t)c->t;
    int rc;
    if (c->algo == SW_ALGO_TILED) {
        rc = sw::tiled_sweep(c->tiled, c->md, c->key, t, c->spins, c->spins_alt, (unsigned long long *)c->labels, c->stream,
                             c->stats_on ? c->stats : nullptr, &c->launches, ev, obs_row);
        if (rc != 0) return fail(SW_ERR_CUDA, "tiled sweep launch failed: %s", cudaGetErrorString(cudaGetLastError()));
        std::swap(c->spins, c->spins_alt);   // spins_alt now holds S^t, the input of this sweep
    } else if (c->algo == SW_ALGO_SMALL) {
        rc = small_sweeps(c, 1, ev);
    } else if (c->algo == SW_ALGO_HAWICK || c->algo == SW_ALGO_KALENTEV) {
        rc = paper_sweep(c, t, ev);
    } else {
        rc = generic_sweep(c, t, ev);
    }
    c->last_algo = c->algo;
    c->have_labels = true;
    if (c->stats_on) c->stat_sweeps += 1;
    c->t += 1;
    return rc;
}

int launch_observables(sw_ctx *c, unsigned long long *dst, bool zero = true)   // dst: one row of OBS_WORDS words
{
    if (zero) CU_TRY(cudaMemsetAsync(dst, 0, 8 * OBS_WORDS, c->stream));
    const size_t work = (c->L % 16 == 0) ? c->N / 16 : c->N;
    const unsigned grid = (unsigned)std::max<size_t>(1, std::min<size_t>((work + 255) / 256, (size_t)c->sms * 4));
    const uint8_t *sp = c->spins;
    cudaError_t e;
    if (c->q <= 2) e = sw::launch_pdl(sw::k_observables<2>, grid, sw::HIST_THREADS, c->stream, c->md, sp, dst);
    else if (c->q <= 4) e = sw::launch_pdl(sw::k_observables<4>, grid, sw::HIST_THREADS, c->stream, c->md, sp, dst);
    else if (c->q <= 8) e = sw::launch_pdl(sw::k_observables<8>, grid, sw::HIST_THREADS, c->stream, c->md, sp, dst);
    else e = sw::launch_pdl(sw::k_observables<16>, grid, sw::HIST_THREADS, c->stream, c->md, sp, dst);
    CU_TRY(e);
    c->launches += 1;
    return SW_OK;
}

int launch_correlation(sw_ctx *c, int r, unsigned long long *dst)   // dst: 16 zeroed words
{
    const size_t work = (c->L % 16 == 0 && r % 4 == 0) ? c->N / 16 : (c->L % 4 == 0) ? c->N / 4 : c->N;
    const unsigned grid = (unsigned)std::max<size_t>(1, std::min<size_t>((work + 255) / 256, (size_t)c->sms * 4));
    const uint8_t *sp = c->spins;
    const uint32_t ur = (uint32_t)r;
    cudaError_t e;
    if (c->q <= 2) e = sw::launch_pdl(sw::k_correlation<2>, grid, sw::HIST_THREADS, c->stream, c->md, sp, ur, dst);
    else if (c->q <= 4) e = sw::launch_pdl(sw::k_correlation<4>, grid, sw::HIST_THREADS, c->stream, c->md, sp, ur, dst);
    else if (c->q <= 8) e = sw::launch_pdl(sw::k_correlation<8>, grid, sw::HIST_THREADS, c->stream, c->md, sp, ur, dst);
    else e = sw::launch_pdl(sw::k_correlation<16>, grid, sw::HIST_THREADS, c->stream, c->md, sp, ur, dst);
    CU_TRY(e);
    c->launches += 1;
    return SW_OK;
}

sw_ctx *create_impl(int L, int q, int model, double T, uint64_t seed, void *ws, size_t bytes, void *stream, bool own)
{
    if (!args_ok(L, q, model) || !(T > 0.0) || !std::isfinite(T)) {
        fail(SW_ERR_ARG, "sw_create: need 2<=L<=%d, 2<=q<=%d, model in {0,1}, finite T>0 (got L=%d q=%d model=%d T=%g)",
             SW_MAX_L, SW_MAX_Q, L, q, model, T);
        return nullptr;
    }
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
        cudaGetLastError();
        fail(SW_ERR_CUDA, "sw_create: no usable CUDA device (this library has no CPU fallback)");
        return nullptr;
    }
    sw_ctx *c = new (std::nothrow) sw_ctx();
    if (!c) { fail(SW_ERR_NOMEM, "sw_create: out of host memory"); return nullptr; }
    if (const char *ds = std::getenv("SW_DUMMY_SMEM")) sw::g_pdl_dynamic_smem = (unsigned)std::atoi(ds);
    c->L = L; c->q = q; c->model = model; c->T = T; c->seed = seed; c->t = 0;
    c->N = (size_t)L * (size_t)L;
    if (cudaGetDevice(&c->device) != cudaSuccess || cudaDeviceGetAttribute(&c->sms, cudaDevAttrMultiProcessorCount, c->device) != cudaSuccess) {
        fail(SW_ERR_CUDA, "sw_create: cannot query the current device: %s", cudaGetErrorString(cudaGetLastError()));
        delete c;
        return nullptr;
    }
    c->cv = carve(L, q);
    if (own) {
        cudaError_t e = cudaMalloc((void **)&c->ws, c->cv.total);
        if (e != cudaSuccess) {
            fail(SW_ERR_NOMEM, "sw_create: cudaMalloc(%zu) failed: %s", c->cv.total, cudaGetErrorString(e));
            delete c;
            return nullptr;
        }
        c->own_ws = true;
        e = cudaStreamCreateWithFlags(&c->stream, cudaStreamNonBlocking);
        if (e != cudaSuccess) {
            fail(SW_ERR_CUDA, "sw_create: cudaStreamCreate failed: %s", cudaGetErrorString(e));
            cudaFree(c->ws);
            delete c;
            return nullptr;
        }
        c->own_stream = true;
    } else {
        if (!ws || bytes < c->cv.total || ((uintptr_t)ws & 255u)) {
            fail(SW_ERR_ARG, "sw_create_in: workspace must be non-NULL, 256-byte aligned and >= %zu bytes (got %zu)",
                 c->cv.total, bytes);
            delete c;
            return nullptr;
        }
        c->ws = (char *)ws;
        c->stream = (cudaStream_t)stream;
    }
    c->spins = (uint8_t *)(c->ws + c->cv.spins);
    c->spins_alt = (uint8_t *)(c->ws + c->cv.spins2);
    c->labels = (int32_t *)(c->ws + c->cv.labels);
    c->labels2 = (int32_t *)(c->ws + c->cv.labels2);
    c->bonds = (uint8_t *)(c->ws + c->cv.bonds);
    c->table = (uint32_t *)(c->ws + c->cv.table);
    c->obs = (unsigned long long *)(c->ws + c->cv.obs);
    c->flag = (int *)(c->ws + c->cv.flag);
    if (const char *ng = std::getenv("SW_NO_GRAPH")) c->graph_off = std::atoi(ng) != 0;
    c->stats = (unsigned long long *)(c->ws + c->cv.stats);
    c->ring = (unsigned long long *)(c->ws + c->cv.ring);
    c->tiled_ws = c->ws + c->cv.tiled;
    c->small_lat = (sw::SmallLattice *)(c->ws + c->cv.small);
    c->key = sw::make_philox_key(seed);
    build_thresholds(c);
    if (cudaMallocHost((void **)&c->rec_host, (size_t)REC_ROWS * OBS_WORDS * 8) != cudaSuccess) {
        fail(SW_ERR_NOMEM, "sw_create: cudaMallocHost failed: %s", cudaGetErrorString(cudaGetLastError()));
        c->rec_host = nullptr;
        sw_destroy(c);
        return nullptr;
    }
    c->md.L = L; c->md.q = q; c->md.model = model; c->md.N = (uint32_t)c->N;
    c->md.thr_potts = (model == SW_POTTS) ? c->thr_host[0] : 0u;
    c->md.table = c->table;

    bool ok = true;
    ok = ok && cudaMemsetAsync(c->table, 0, 4 * (size_t)(2 * SW_MAX_Q) * (2 * SW_MAX_Q), c->stream) == cudaSuccess;
    if (model == SW_CLOCK)
        ok = ok && cudaMemcpyAsync(c->table, c->thr_host.data(), 4 * c->thr_host.size(), cudaMemcpyHostToDevice, c->stream) == cudaSuccess;
    ok = ok && cudaMemsetAsync(c->stats, 0, 8 * SW_NUM_STATS, c->stream) == cudaSuccess;
    {
        sw::SmallLattice sl;
        sl.key = c->key;
        sl.thr_potts = c->md.thr_potts;
        sl.pad = 0u;
        ok = ok && cudaMemcpyAsync(c->small_lat, &sl, sizeof(sl), cudaMemcpyHostToDevice, c->stream) == cudaSuccess;
        ok = ok && cudaStreamSynchronize(c->stream) == cudaSuccess;     // sl is on the stack
    }
    if (ok) {
        sw::k_init_spins<<<blocks_for((c->N + 3) / 4, 256), 256, 0, c->stream>>>(c->md, c->key, c->spins);
        c->launches += 1;
        ok = cudaGetLastError() == cudaSuccess;
    }
    c->algo = auto_algo(L);
    if (ok && sw::tiled_supported(L)) ok = sw::tiled_init(c->tiled, c->md, c->tiled_ws, c->spins, c->spins_alt) == 0;
    ok = ok && cudaStreamSynchronize(c->stream) == cudaSuccess;
    if (!ok) {
        fail(SW_ERR_CUDA, "sw_create: device initialisation failed: %s", cudaGetErrorString(cudaGetLastError()));
        sw_destroy(c);
        return nullptr;
    }
    return c;
}

}  // namespace

extern "C" {

size_t sw_workspace_bytes(int L, int q, int model)
{
    if (!args_ok(L, q, model)) return 0;
    return carve(L, q).total;
}

sw_ctx *sw_create(int L, int q, int model, double T, uint64_t seed)
{
    return create_impl(L, q, model, T, seed, nullptr, 0, nullptr, true);
}

sw_ctx *sw_create_in(int L, int q, int model, double T, uint64_t seed, void *d_workspace, size_t bytes, void *cuda_stream)
{
    return create_impl(L, q, model, T, seed, d_workspace, bytes, cuda_stream, false);
}

void sw_destroy(sw_ctx *c)
{
    if (!c) return;
    DeviceGuard guard(c);
    if (c->stream || !c->own_stream) cudaStreamSynchronize(c->stream);
    if (c->rec_host) cudaFreeHost(c->rec_host);
    for (int k = 0; k < 2; ++k) {
        if (c->graph[k].exec) cudaGraphExecDestroy(c->graph[k].exec);
        if (c->graph[k].graph) cudaGraphDestroy(c->graph[k].graph);
    }
    if (c->own_ws && c->ws) cudaFree(c->ws);
    if (c->own_stream && c->stream) cudaStreamDestroy(c->stream);
    delete c;
}

int sw_sweep_async(sw_ctx *c, int n)
{
    if (!c || n < 0) return fail(SW_ERR_ARG, "sw_sweep: NULL context or n < 0");
    DeviceGuard guard(c);
    if (c->t + (uint64_t)n > 0xFFFFFFFFull) return fail(SW_ERR_ARG, "sw_sweep: sweep index would exceed 2^32-1");
    if (c->algo == SW_ALGO_SMALL && n > 0) {       // all n sweeps inside one launch
        int rc = small_sweeps(c, n);
        if (rc != SW_OK) return rc;
        c->last_algo = c->algo;
        c->have_labels = true;
        if (c->stats_on) c->stat_sweeps += (uint64_t)n;
        c->t += (uint64_t)n;
        n = 0;
    }
    if (c->algo == SW_ALGO_TILED && !c->stats_on) n -= graph_sweeps(c, n);
    for (int k = 0; k < n; ++k) {
        int rc = one_sweep(c);
        if (rc != SW_OK) return rc;
    }
    CU_TRY(cudaGetLastError());
    return SW_OK;
}

int sw_sync(sw_ctx *c)
{
    if (!c) return fail(SW_ERR_ARG, "sw_sync: NULL context");
    DeviceGuard guard(c);
    CU_TRY(cudaStreamSynchronize(c->stream));
    return SW_OK;
}

int sw_sweep(sw_ctx *c, int n)
{
    int rc = sw_sweep_async(c, n);
    if (rc != SW_OK) return rc;
    return sw_sync(c);
}

namespace {
// n sweeps, row k of every output = the configuration BEFORE the k-th sweep of the call (R10).
// r1 < 0: no correlation histograms.
int record_impl(sw_ctx *c, int n, int r1, int r2, int64_t *bond_out, int64_t *state_out, int64_t *c1_out, int64_t *c2_out)
{
    unsigned long long *host = c->rec_host;   // pinned staging buffer of the ring (allocated with the context)
    const bool fused = fuses_observables(c);
    int done = 0;
    while (done < n) {
        const int chunk = std::min(REC_ROWS, n - done);
        CU_TRY(cudaMemsetAsync(c->ring, 0, (size_t)chunk * OBS_WORDS * 8, c->stream));   // all rows of the chunk at once
        for (int k = 0; k < chunk; ++k) {
            unsigned long long *row = c->ring + (size_t)k * OBS_WORDS;
            int rc = fused ? SW_OK : launch_observables(c, row, false);
            if (rc != SW_OK) return rc;
            if (r1 >= 0) {
                rc = launch_correlation(c, r1, row + 32);
                if (rc == SW_OK) rc = launch_correlation(c, r2, row + 48);
                if (rc != SW_OK) return rc;
            }
            rc = one_sweep(c, nullptr, fused ? row : nullptr);
            if (rc != SW_OK) return rc;
        }
        CU_TRY(cudaGetLastError());
        CU_TRY(cudaMemcpyAsync(host, c->ring, (size_t)chunk * OBS_WORDS * 8, cudaMemcpyDeviceToHost, c->stream));
        CU_TRY(cudaStreamSynchronize(c->stream));
        for (int k = 0; k < chunk; ++k)
            for (int j = 0; j < c->q; ++j) {
                const size_t o = (size_t)(done + k) * c->q + j;
                bond_out[o] = (int64_t)host[(size_t)k * OBS_WORDS + j];
                state_out[o] = (int64_t)host[(size_t)k * OBS_WORDS + 16 + j];
                if (r1 >= 0) {
                    c1_out[o] = (int64_t)host[(size_t)k * OBS_WORDS + 32 + j];
                    c2_out[o] = (int64_t)host[(size_t)k * OBS_WORDS + 48 + j];
                }
            }
        done += chunk;
    }
    return SW_OK;
}
}  // namespace

int sw_sweep_record(sw_ctx *c, int n, int64_t *bond_out, int64_t *state_out)
{
    if (!c || n < 0 || !bond_out || !state_out) return fail(SW_ERR_ARG, "sw_sweep_record: bad arguments");
    DeviceGuard guard(c);
    if (c->t + (uint64_t)n > 0xFFFFFFFFull) return fail(SW_ERR_ARG, "sw_sweep_record: sweep index would exceed 2^32-1");
    return record_impl(c, n, -1, -1, bond_out, state_out, nullptr, nullptr);
}

int sw_sweep_record_corr(sw_ctx *c, int n, int r1, int r2, int64_t *bond_out, int64_t *state_out, int64_t *corr1_out,
                         int64_t *corr2_out)
{
    if (!c || n < 0 || !bond_out || !state_out || !corr1_out || !corr2_out || r1 < 0 || r2 < 0 || r1 >= c->L || r2 >= c->L)
        return fail(SW_ERR_ARG, "sw_sweep_record_corr: bad arguments (need 0 <= r1, r2 < L and non-NULL outputs)");
    DeviceGuard guard(c);
    if (c->t + (uint64_t)n > 0xFFFFFFFFull) return fail(SW_ERR_ARG, "sw_sweep_record_corr: sweep index would exceed 2^32-1");
    return record_impl(c, n, r1, r2, bond_out, state_out, corr1_out, corr2_out);
}

int sw_correlation(sw_ctx *c, int r, int64_t *corr_hist)
{
    if (!c || !corr_hist || r < 0 || r >= c->L) return fail(SW_ERR_ARG, "sw_correlation: need 0 <= r < L and a non-NULL output");
    DeviceGuard guard(c);
    CU_TRY(cudaMemsetAsync(c->obs, 0, 8 * OBS_WORDS, c->stream));
    int rc = launch_correlation(c, r, c->obs + 32);
    if (rc != SW_OK) return rc;
    CU_TRY(cudaGetLastError());
    unsigned long long host[16];
    CU_TRY(cudaMemcpyAsync(host, c->obs + 32, sizeof(host), cudaMemcpyDeviceToHost, c->stream));
    CU_TRY(cudaStreamSynchronize(c->stream));
    for (int j = 0; j < c->q; ++j) corr_hist[j] = (int64_t)host[j];
    return SW_OK;
}

int sw_observables(sw_ctx *c, int64_t *bond_hist, int64_t *state_hist)
{
    if (!c || !bond_hist || !state_hist) return fail(SW_ERR_ARG, "sw_observables: NULL argument");
    DeviceGuard guard(c);
    int rc = launch_observables(c, c->obs);
    if (rc != SW_OK) return rc;
    CU_TRY(cudaGetLastError());
    unsigned long long host[OBS_WORDS];
    CU_TRY(cudaMemcpyAsync(host, c->obs, sizeof(host), cudaMemcpyDeviceToHost, c->stream));
    CU_TRY(cudaStreamSynchronize(c->stream));
    for (int j = 0; j < c->q; ++j) {
        bond_hist[j] = (int64_t)host[j];
        state_hist[j] = (int64_t)host[16 + j];
    }
    return SW_OK;
}

int sw_get_spins(sw_ctx *c, uint8_t *host_out)
{
    if (!c || !host_out) return fail(SW_ERR_ARG, "sw_get_spins: NULL argument");
    DeviceGuard guard(c);
    CU_TRY(cudaMemcpyAsync(host_out, c->spins, c->N, cudaMemcpyDeviceToHost, c->stream));
    CU_TRY(cudaStreamSynchronize(c->stream));
    return SW_OK;
}

int sw_set_spins(sw_ctx *c, const uint8_t *host_in, uint64_t sweep_index)
{
    if (!c || !host_in) return fail(SW_ERR_ARG, "sw_set_spins: NULL argument");
    DeviceGuard guard(c);
    if (sweep_index > 0xFFFFFFFFull) return fail(SW_ERR_ARG, "sw_set_spins: sweep index must fit 32 bits");
    // Stage in the bond scratch buffer, validate on the device, then commit.
    CU_TRY(cudaMemcpyAsync(c->bonds, host_in, c->N, cudaMemcpyHostToDevice, c->stream));
    CU_TRY(cudaMemsetAsync(c->flag, 0, sizeof(int), c->stream));
    sw::k_check_spins<<<blocks_for(c->N, 256), 256, 0, c->stream>>>(c->md.N, (uint32_t)c->q, c->bonds, c->flag);
    c->launches += 1;
    CU_TRY(cudaGetLastError());
    int bad = 0;
    CU_TRY(cudaMemcpyAsync(&bad, c->flag, sizeof(int), cudaMemcpyDeviceToHost, c->stream));
    CU_TRY(cudaStreamSynchronize(c->stream));
    if (bad) return fail(SW_ERR_ARG, "sw_set_spins: a spin value is >= q = %d", c->q);
    CU_TRY(cudaMemcpyAsync(c->spins, c->bonds, c->N, cudaMemcpyDeviceToDevice, c->stream));
    CU_TRY(cudaStreamSynchronize(c->stream));
    c->t = sweep_index;
    c->have_labels = false;
    return SW_OK;
}

uint64_t sw_sweep_index(sw_ctx *c) { return c ? c->t : 0; }

int sw_get_thresholds(sw_ctx *c, uint32_t *out, int *count)
{
    if (!c || !count) return fail(SW_ERR_ARG, "sw_get_thresholds: NULL argument");
    *count = (int)c->thr_host.size();
    if (out) std::memcpy(out, c->thr_host.data(), 4 * c->thr_host.size());
    return SW_OK;
}

int sw_get_labels(sw_ctx *c, int32_t *host_out)
{
    if (!c || !host_out) return fail(SW_ERR_ARG, "sw_get_labels: NULL argument");
    DeviceGuard guard(c);
    if (!c->have_labels) return fail(SW_ERR_ARG, "sw_get_labels: no sweep has been executed on this configuration");
    if (c->last_algo == SW_ALGO_TILED) {
        // The tiled sweep fuses the decisions of tile-local clusters into its labels, so the canonical roots are
        // rebuilt from the sweep's input (still in the other ping-pong buffer) and its bonds (sweep index t - 1).
        // No allocation: the union-find nodes take the first N/2 bytes of the 4N-byte label array, the resolved labels
        // are staged behind them, half of the lattice (2N bytes) at a time.
        unsigned long long *parent = (unsigned long long *)c->labels;
        int32_t *stage = c->labels + c->N / 4;           // byte offset N: past the N/2 bytes of nodes, 1024-aligned
        if (sw::tiled_relabel(c->tiled, c->md, c->key, (uint32_t)(c->t - 1), c->spins_alt, parent, c->stream, &c->launches) != 0)
            return fail(SW_ERR_CUDA, "sw_get_labels: relabel launch failed: %s", cudaGetErrorString(cudaGetLastError()));
        const uint32_t half = (uint32_t)(c->N / 2);
        for (uint32_t part = 0; part < 2; ++part) {
            if (sw::tiled_resolve_chunk(c->tiled, c->md, parent, part * half, half, stage, c->stream, &c->launches) != 0)
                return fail(SW_ERR_CUDA, "sw_get_labels: resolve launch failed: %s", cudaGetErrorString(cudaGetLastError()));
            CU_TRY(cudaMemcpyAsync(host_out + (size_t)part * half, stage, 4 * (size_t)half, cudaMemcpyDeviceToHost, c->stream));
            CU_TRY(cudaStreamSynchronize(c->stream));
        }
        return SW_OK;
    }
    CU_TRY(cudaGetLastError());
    CU_TRY(cudaMemcpyAsync(host_out, c->labels, 4 * c->N, cudaMemcpyDeviceToHost, c->stream));
    CU_TRY(cudaStreamSynchronize(c->stream));
    return SW_OK;
}

int sw_debug_bonds(sw_ctx *c, uint8_t *host_out)
{
    if (!c || !host_out) return fail(SW_ERR_ARG, "sw_debug_bonds: NULL argument");
    DeviceGuard guard(c);
    sw::k_bonds<<<blocks_for((c->N + 1) / 2, 256), 256, 0, c->stream>>>(c->md, c->key, (uint32_t)c->t, c->spins, c->bonds);
    c->launches += 1;
    CU_TRY(cudaGetLastError());
    CU_TRY(cudaMemcpyAsync(host_out, c->bonds, c->N, cudaMemcpyDeviceToHost, c->stream));
    CU_TRY(cudaStreamSynchronize(c->stream));
    return SW_OK;
}

int sw_set_algorithm(sw_ctx *c, int algo)
{
    if (!c) return fail(SW_ERR_ARG, "sw_set_algorithm: NULL context");
    if (algo == SW_ALGO_AUTO) algo = auto_algo(c->L);
    if (algo == SW_ALGO_TILED && !sw::tiled_supported(c->L))
        return fail(SW_ERR_UNSUPPORTED, "sw_set_algorithm: the tiled back-end needs L %% %d == 0 (L = %d)", sw::TW, c->L);
    if (algo == SW_ALGO_SMALL && !sw::small_supported(c->L))
        return fail(SW_ERR_UNSUPPORTED, "sw_set_algorithm: the one-CTA back-end needs L <= %d (L = %d)", sw::SMALL_MAX_L, c->L);
    if (algo != SW_ALGO_GENERIC && algo != SW_ALGO_TILED && algo != SW_ALGO_SMALL && algo != SW_ALGO_HAWICK && algo != SW_ALGO_KALENTEV)
        return fail(SW_ERR_ARG, "sw_set_algorithm: unknown back-end %d", algo);
    c->algo = algo;
    return SW_OK;
}

int sw_get_algorithm(sw_ctx *c) { return c ? c->algo : SW_ERR_ARG; }

int sw_enable_stats(sw_ctx *c, int on)
{
    if (!c) return fail(SW_ERR_ARG, "sw_enable_stats: NULL context");
    c->stats_on = on != 0;
    return SW_OK;
}

int sw_stats(sw_ctx *c, double *out4)
{
    if (!c || !out4) return fail(SW_ERR_ARG, "sw_stats: NULL argument");
    DeviceGuard guard(c);
    unsigned long long h[SW_NUM_STATS];
    CU_TRY(cudaMemcpyAsync(h, c->stats, sizeof(h), cudaMemcpyDeviceToHost, c->stream));
    CU_TRY(cudaStreamSynchronize(c->stream));
    for (int k = 0; k < SW_NUM_STATS; ++k) out4[k] = (double)h[k];
    out4[0] = (double)c->stat_sweeps;
    out4[5] = (double)c->ccl_iterations;
    out4[6] = (double)c->ccl_sweeps;
    out4[7] = (double)c->graph_replays;
    return SW_OK;
}

int sw_sweep_profile(sw_ctx *c, int n, double *ms_out, int *n_kernels)
{
    if (!c || n < 0 || !ms_out || !n_kernels) return fail(SW_ERR_ARG, "sw_sweep_profile: bad arguments");
    DeviceGuard guard(c);
    if (c->t + (uint64_t)n > 0xFFFFFFFFull) return fail(SW_ERR_ARG, "sw_sweep_profile: sweep index would exceed 2^32-1");
    const int nk = (c->algo == SW_ALGO_TILED) ? sw::TILED_NUM_KERNELS : (c->algo == SW_ALGO_SMALL) ? 1 :
                   (c->algo == SW_ALGO_HAWICK || c->algo == SW_ALGO_KALENTEV) ? 3 : 5;
    cudaEvent_t ev[SW_MAX_KERNELS + 1];
    for (int k = 0; k <= nk; ++k) CU_TRY(cudaEventCreate(&ev[k]));
    for (int k = 0; k < SW_MAX_KERNELS; ++k) ms_out[k] = 0.0;
    int rc = SW_OK;
    for (int it = 0; it < n && rc == SW_OK; ++it) {
        rc = one_sweep(c, ev);
        if (rc != SW_OK) break;
        if (cudaStreamSynchronize(c->stream) != cudaSuccess) { rc = fail(SW_ERR_CUDA, "sw_sweep_profile: sync failed"); break; }
        for (int k = 0; k < nk; ++k) {
            float ms = 0.f;
            cudaEventElapsedTime(&ms, ev[k], ev[k + 1]);
            ms_out[k] += (double)ms;
        }
    }
    for (int k = 0; k <= nk; ++k) cudaEventDestroy(ev[k]);
    *n_kernels = nk;
    return rc;
}

const char *sw_kernel_name(sw_ctx *c, int k)
{
    if (!c || k < 0) return nullptr;
    if (c->algo == SW_ALGO_TILED) return k < sw::TILED_NUM_KERNELS ? sw::TILED_KERNELS[k] : nullptr;
    if (c->algo == SW_ALGO_SMALL) return k == 0 ? "k_small_sweeps" : nullptr;
    if (c->algo == SW_ALGO_HAWICK || c->algo == SW_ALGO_KALENTEV) {
        static const char *const names[3] = { "k_bonds", "label equivalence (all iterations)", "k_flip" };
        return k < 3 ? names[k] : nullptr;
    }
    return k < 5 ? GENERIC_KERNELS[k] : nullptr;
}

uint64_t sw_launch_count(sw_ctx *c) { return c ? c->launches : 0; }

// ---------------------------------------------------------------------------------------------------------------
// Batches of independent lattices (NEXT-2): same L, q, model; own temperature and seed each.
// ---------------------------------------------------------------------------------------------------------------
}  // extern "C"

struct sw_batch {
    int B = 0, L = 0, q = 0, model = 0, device = 0, sms = 148;
    size_t N = 0;
    uint64_t t = 0;
    cudaStream_t stream = nullptr;
    char *ws = nullptr;
    uint8_t *spins = nullptr;            // [B][N]
    sw::SmallLattice *lats = nullptr;    // [B]
    uint32_t *tables = nullptr;          // [B][SMALL_TABLE_WORDS] (clock)
    unsigned long long *obs = nullptr;   // [B][OBS_WORDS]
    std::vector<sw::Model> md;           // per lattice (host)
    // L % 128 == 0: the tiled kernels over the tiles of all lattices (spins ping-pong, labels, union-find nodes)
    bool tiled = false;
    uint8_t *spins_alt = nullptr;        // [B][N]
    unsigned long long *parent = nullptr;
    sw::PhiloxKey *keys = nullptr;       // [B]
    uint32_t *thr = nullptr;             // [B]
    sw::TiledState st{};
    uint64_t launches = 0;
};

namespace {
struct BatchGuard {
    int prev = -1;
    bool switched = false;
    explicit BatchGuard(const sw_batch *b)
    {
        if (b && cudaGetDevice(&prev) == cudaSuccess && prev != b->device) switched = cudaSetDevice(b->device) == cudaSuccess;
    }
    ~BatchGuard() { if (switched) cudaSetDevice(prev); }
};
}  // namespace

extern "C" {

sw_batch *sw_create_batch(int B, int L, int q, int model, const double *T, const uint64_t *seed)
{
    if (B < 1 || B > SW_MAX_BATCH || !T || !seed || !args_ok(L, q, model)) {
        fail(SW_ERR_ARG, "sw_create_batch: need 1 <= B <= %d, valid L, q, model and non-NULL T, seed", SW_MAX_BATCH);
        return nullptr;
    }
    for (int b = 0; b < B; ++b)
        if (!(T[b] > 0.0) || !std::isfinite(T[b])) {
            fail(SW_ERR_ARG, "sw_create_batch: T[%d] = %g is not a finite positive temperature", b, T[b]);
            return nullptr;
        }
    const bool tiled = sw::tiled_supported(L);      // measured: 0.008 ns per flip through the tiles, 0.03 through one CTA per lattice
    if (!tiled && !sw::small_supported(L)) {
        fail(SW_ERR_UNSUPPORTED, "sw_create_batch: L = %d: batches need L <= %d (one CTA per lattice) or L %% %d == 0 (tiles)", L,
             sw::SMALL_MAX_L, sw::TW);
        return nullptr;
    }
    if (tiled && (size_t)B * (size_t)(L / sw::TW) * (size_t)(L / sw::TH) * sw::OCAP >= (1ull << 32)) {
        fail(SW_ERR_ARG, "sw_create_batch: B * tiles too large for 32-bit union-find nodes");
        return nullptr;
    }
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
        cudaGetLastError();
        fail(SW_ERR_CUDA, "sw_create_batch: no usable CUDA device (this library has no CPU fallback)");
        return nullptr;
    }
    sw_batch *bt = new (std::nothrow) sw_batch();
    if (!bt) { fail(SW_ERR_NOMEM, "sw_create_batch: out of host memory"); return nullptr; }
    bt->B = B; bt->L = L; bt->q = q; bt->model = model; bt->N = (size_t)L * L;
    cudaGetDevice(&bt->device);
    cudaDeviceGetAttribute(&bt->sms, cudaDevAttrMultiProcessorCount, bt->device);
    bt->tiled = tiled;
    const size_t tiles = tiled ? (size_t)(L / sw::TW) * (L / sw::TH) : 0;
    const size_t o_spins = 0, o_lats = align_up((size_t)B * bt->N), o_tab = o_lats + align_up((size_t)B * sizeof(sw::SmallLattice)),
                 o_obs = o_tab + align_up((size_t)B * sw::SMALL_TABLE_WORDS * 4), o_alt = o_obs + align_up((size_t)B * OBS_WORDS * 8),
                 o_par = o_alt + (tiled ? align_up((size_t)B * bt->N) : 0), o_keys = o_par + align_up((size_t)B * tiles * sw::OCAP * 8),
                 o_thr = o_keys + align_up((size_t)B * sizeof(sw::PhiloxKey)), o_tw = o_thr + align_up((size_t)B * 4),
                 total = o_tw + (tiled ? align_up(sw::tiled_workspace_bytes_n(L, (size_t)B)) : 0);
    bool ok = cudaMalloc((void **)&bt->ws, total) == cudaSuccess;
    ok = ok && cudaStreamCreateWithFlags(&bt->stream, cudaStreamNonBlocking) == cudaSuccess;
    if (!ok) {
        fail(SW_ERR_NOMEM, "sw_create_batch: device allocation of %zu bytes failed: %s", total, cudaGetErrorString(cudaGetLastError()));
        sw_batch_destroy(bt);
        return nullptr;
    }
    bt->spins = (uint8_t *)(bt->ws + o_spins);
    bt->lats = (sw::SmallLattice *)(bt->ws + o_lats);
    bt->tables = (uint32_t *)(bt->ws + o_tab);
    bt->obs = (unsigned long long *)(bt->ws + o_obs);
    bt->spins_alt = (uint8_t *)(bt->ws + o_alt);
    bt->parent = (unsigned long long *)(bt->ws + o_par);
    bt->keys = (sw::PhiloxKey *)(bt->ws + o_keys);
    bt->thr = (uint32_t *)(bt->ws + o_thr);
    // per-lattice thresholds (host, double: R1 / R4, R6, R7) and Philox keys; S^0 of every lattice from its INIT stream
    std::vector<sw::SmallLattice> hl((size_t)B);
    std::vector<uint32_t> ht((size_t)B * sw::SMALL_TABLE_WORDS, 0u);
    bt->md.resize((size_t)B);
    sw_ctx tmp;
    tmp.q = q; tmp.model = model;
    for (int b = 0; b < B; ++b) {
        tmp.T = T[b];
        build_thresholds(&tmp);
        hl[b].key = sw::make_philox_key(seed[b]);
        hl[b].thr_potts = model == SW_POTTS ? tmp.thr_host[0] : 0u;
        hl[b].pad = 0u;
        if (model == SW_CLOCK) std::copy(tmp.thr_host.begin(), tmp.thr_host.end(), ht.begin() + (size_t)b * sw::SMALL_TABLE_WORDS);
        sw::Model &m = bt->md[b];
        m.L = L; m.q = q; m.model = model; m.N = (uint32_t)bt->N; m.thr_potts = hl[b].thr_potts;
        m.table = bt->tables + (size_t)b * sw::SMALL_TABLE_WORDS;
    }
    ok = cudaMemcpyAsync(bt->lats, hl.data(), hl.size() * sizeof(sw::SmallLattice), cudaMemcpyHostToDevice, bt->stream) == cudaSuccess;
    ok = ok && cudaMemcpyAsync(bt->tables, ht.data(), ht.size() * 4, cudaMemcpyHostToDevice, bt->stream) == cudaSuccess;
    std::vector<sw::PhiloxKey> hk((size_t)B);
    std::vector<uint32_t> hthr((size_t)B);
    if (tiled) {
        for (int b = 0; b < B; ++b) { hk[b] = hl[b].key; hthr[b] = hl[b].thr_potts; }
        ok = ok && cudaMemcpyAsync(bt->keys, hk.data(), hk.size() * sizeof(sw::PhiloxKey), cudaMemcpyHostToDevice, bt->stream) == cudaSuccess;
        ok = ok && cudaMemcpyAsync(bt->thr, hthr.data(), hthr.size() * 4, cudaMemcpyHostToDevice, bt->stream) == cudaSuccess;
        ok = ok && sw::tiled_init(bt->st, bt->md[0], bt->ws + o_tw, bt->spins, bt->spins_alt, (size_t)B) == 0;
        bt->st.batch = true;
        bt->st.bv.keys = bt->keys;
        bt->st.bv.thr = bt->thr;
        bt->st.bv.tables = bt->tables;
    }
    for (int b = 0; b < B && ok; ++b) {
        sw::k_init_spins<<<blocks_for((bt->N + 3) / 4, 256), 256, 0, bt->stream>>>(bt->md[b], hl[b].key, bt->spins + (size_t)b * bt->N);
        ok = cudaGetLastError() == cudaSuccess;
    }
    ok = ok && cudaStreamSynchronize(bt->stream) == cudaSuccess;
    if (!ok) {
        fail(SW_ERR_CUDA, "sw_create_batch: device initialisation failed: %s", cudaGetErrorString(cudaGetLastError()));
        sw_batch_destroy(bt);
        return nullptr;
    }
    return bt;
}

void sw_batch_destroy(sw_batch *bt)
{
    if (!bt) return;
    BatchGuard guard(bt);
    if (bt->stream) { cudaStreamSynchronize(bt->stream); cudaStreamDestroy(bt->stream); }
    if (bt->ws) cudaFree(bt->ws);
    delete bt;
}

int sw_batch_sweep(sw_batch *bt, int n)
{
    if (!bt || n < 0) return fail(SW_ERR_ARG, "sw_batch_sweep: NULL batch or n < 0");
    if (bt->t + (uint64_t)n > 0xFFFFFFFFull) return fail(SW_ERR_ARG, "sw_batch_sweep: sweep index would exceed 2^32-1");
    BatchGuard guard(bt);
    if (n > 0 && !bt->tiled) {
        CU_TRY(sw::small_launch(bt->model, bt->B, bt->L, bt->q, bt->lats, bt->tables, bt->spins, nullptr, (uint32_t)bt->t, n, bt->stream));
        bt->t += (uint64_t)n;
    } else {
        for (int k = 0; k < n; ++k) {      // three launches per sweep for the whole batch
            if (sw::tiled_sweep(bt->st, bt->md[0], sw::PhiloxKey{}, (uint32_t)bt->t, bt->spins, bt->spins_alt, bt->parent, bt->stream, nullptr,
                                &bt->launches, nullptr) != 0)
                return fail(SW_ERR_CUDA, "sw_batch_sweep: launch failed: %s", cudaGetErrorString(cudaGetLastError()));
            std::swap(bt->spins, bt->spins_alt);
            bt->t += 1;
        }
    }
    CU_TRY(cudaStreamSynchronize(bt->stream));
    return SW_OK;
}

int sw_batch_get_spins(sw_batch *bt, uint8_t *host_out)
{
    if (!bt || !host_out) return fail(SW_ERR_ARG, "sw_batch_get_spins: NULL argument");
    BatchGuard guard(bt);
    CU_TRY(cudaMemcpyAsync(host_out, bt->spins, (size_t)bt->B * bt->N, cudaMemcpyDeviceToHost, bt->stream));
    CU_TRY(cudaStreamSynchronize(bt->stream));
    return SW_OK;
}

int sw_batch_set_spins(sw_batch *bt, const uint8_t *host_in, uint64_t sweep_index)
{
    if (!bt || !host_in) return fail(SW_ERR_ARG, "sw_batch_set_spins: NULL argument");
    if (sweep_index > 0xFFFFFFFFull) return fail(SW_ERR_ARG, "sw_batch_set_spins: sweep index must fit 32 bits");
    const size_t total = (size_t)bt->B * bt->N;
    for (size_t i = 0; i < total; ++i)
        if (host_in[i] >= (uint8_t)bt->q) return fail(SW_ERR_ARG, "sw_batch_set_spins: spin value %d >= q = %d", (int)host_in[i], bt->q);
    BatchGuard guard(bt);
    CU_TRY(cudaMemcpyAsync(bt->spins, host_in, total, cudaMemcpyHostToDevice, bt->stream));
    CU_TRY(cudaStreamSynchronize(bt->stream));
    bt->t = sweep_index;
    return SW_OK;
}

int sw_batch_observables(sw_batch *bt, int64_t *bond_hist, int64_t *state_hist)
{
    if (!bt || !bond_hist || !state_hist) return fail(SW_ERR_ARG, "sw_batch_observables: NULL argument");
    BatchGuard guard(bt);
    CU_TRY(cudaMemsetAsync(bt->obs, 0, (size_t)bt->B * OBS_WORDS * 8, bt->stream));
    const size_t work = (bt->L % 16 == 0) ? bt->N / 16 : bt->N;
    const unsigned grid = (unsigned)std::max<size_t>(1, std::min<size_t>((work + 255) / 256, (size_t)bt->sms * 4));
    for (int b = 0; b < bt->B; ++b) {
        const uint8_t *sp = bt->spins + (size_t)b * bt->N;
        unsigned long long *dst = bt->obs + (size_t)b * OBS_WORDS;
        cudaError_t e;
        if (bt->q <= 2) e = sw::launch_pdl(sw::k_observables<2>, grid, sw::HIST_THREADS, bt->stream, bt->md[b], sp, dst);
        else if (bt->q <= 4) e = sw::launch_pdl(sw::k_observables<4>, grid, sw::HIST_THREADS, bt->stream, bt->md[b], sp, dst);
        else if (bt->q <= 8) e = sw::launch_pdl(sw::k_observables<8>, grid, sw::HIST_THREADS, bt->stream, bt->md[b], sp, dst);
        else e = sw::launch_pdl(sw::k_observables<16>, grid, sw::HIST_THREADS, bt->stream, bt->md[b], sp, dst);
        CU_TRY(e);
    }
    std::vector<unsigned long long> host((size_t)bt->B * OBS_WORDS);
    CU_TRY(cudaMemcpyAsync(host.data(), bt->obs, host.size() * 8, cudaMemcpyDeviceToHost, bt->stream));
    CU_TRY(cudaStreamSynchronize(bt->stream));
    for (int b = 0; b < bt->B; ++b)
        for (int j = 0; j < bt->q; ++j) {
            bond_hist[(size_t)b * bt->q + j] = (int64_t)host[(size_t)b * OBS_WORDS + j];
            state_hist[(size_t)b * bt->q + j] = (int64_t)host[(size_t)b * OBS_WORDS + 16 + j];
        }
    return SW_OK;
}

uint64_t sw_batch_sweep_index(sw_batch *bt) { return bt ? bt->t : 0; }

int sw_selftest(void)
{
    static const uint32_t base[] = { 0u, 1u, 2u, 0x7FFFFFFFu, 0x80000000u, 0x80000001u, 0x95F61998u, 0xAAAAAAAAu, 0xFFFFFFFEu, 0xFFFFFFFFu };
    std::vector<uint32_t> v(base, base + sizeof(base) / sizeof(base[0]));
    for (uint32_t k = 0; k < 54; ++k) v.push_back(0x9E3779B9u * (k + 1u) + (k << 27));
    for (size_t k = 0, n0 = v.size(); k < n0; ++k) { v.push_back(v[k] + 1u); v.push_back(v[k] - 1u); }
    const int n = (int)v.size();
    uint32_t *d_v = nullptr;
    int *d_bad = nullptr;
    CU_TRY(cudaMalloc((void **)&d_v, 4 * (size_t)n));
    cudaError_t e = cudaMalloc((void **)&d_bad, 2 * sizeof(int));
    if (e != cudaSuccess) { cudaFree(d_v); return fail(SW_ERR_NOMEM, "sw_selftest: cudaMalloc failed"); }
    int bad[2] = { -1, -1 };
    e = cudaMemcpy(d_v, v.data(), 4 * (size_t)n, cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemset(d_bad, 0, 2 * sizeof(int));
    if (e == cudaSuccess) {
        sw::k_selftest_compare<<<(n * n + 255) / 256, 256>>>(d_v, n, d_bad);
        e = cudaGetLastError();
    }
    if (e == cudaSuccess) e = cudaMemcpy(bad, d_bad, sizeof(bad), cudaMemcpyDeviceToHost);
    cudaFree(d_v);
    cudaFree(d_bad);
    if (e != cudaSuccess) return fail(SW_ERR_CUDA, "sw_selftest: %s", cudaGetErrorString(e));
    if (bad[0] || bad[1])
        return fail(SW_ERR_UNSUPPORTED, "sw_selftest: carry-flag compares disagree with >= (sub form %d, add form %d of %d pairs)", bad[0], bad[1], n * n);
    return SW_OK;
}

const char *sw_last_error(void) { return g_err; }

}  // extern "C"

// ---------------------------------------------------------------------------------------------------------------------
// sw_sweep_noalloc (include/sw.h): one sweep of the generic back-end whose scratch is a static device array, for callers
// that cannot call cudaMalloc.  No existing path uses anything below.
// ---------------------------------------------------------------------------------------------------------------------
#include <mutex>

namespace {

constexpr size_t NOALLOC_MAX_N = (size_t)SW_NOALLOC_MAX_L * SW_NOALLOC_MAX_L;
constexpr size_t NOALLOC_TABLE_BYTES = 4 * (size_t)(2 * SW_MAX_Q) * (2 * SW_MAX_Q);   // 4096: clock thresholds, (2q)^2 words
constexpr size_t NOALLOC_LABELS_OFF = NOALLOC_TABLE_BYTES;                            // int32 parents, 4 bytes per site
constexpr size_t NOALLOC_BONDS_OFF = NOALLOC_LABELS_OFF + 4 * NOALLOC_MAX_N;          // bond bits, 1 byte per site
constexpr size_t NOALLOC_BYTES = NOALLOC_BONDS_OFF + NOALLOC_MAX_N;                   // 5 MiB + 4 KiB

}  // namespace

// The scratch.  In HOST code this name is only a stand-in for the symbol (not a device address): the host takes the
// address once per device with cudaGetSymbolAddress (noalloc_scratch) and hands that pointer to the kernels.
// The table comes first: a threshold lookup with an (unchecked) spin value >= q lands at most
// 4 * ((2*255 + 2q)*2q + 2*255 + 2q) < 72 KB past its start, inside the array.
static __device__ __align__(256) unsigned char g_noalloc_scratch[NOALLOC_BYTES];

namespace {

constexpr int NOALLOC_MAX_DEVICES = 64;
std::mutex g_noalloc_mutex;
unsigned char *g_noalloc_ptr[NOALLOC_MAX_DEVICES] = {};   // device address of g_noalloc_scratch, per device ordinal

// The device address of the scratch on the CURRENT device (looked up on the first call per device, with that device current).
int noalloc_scratch(int dev, unsigned char **out)
{
    std::lock_guard<std::mutex> lock(g_noalloc_mutex);
    if (!g_noalloc_ptr[dev]) {
        void *p = nullptr;
        CU_TRY(cudaGetSymbolAddress(&p, g_noalloc_scratch));
        if (!p) return fail(SW_ERR_CUDA, "sw_sweep_noalloc: cudaGetSymbolAddress returned NULL on device %d", dev);
        g_noalloc_ptr[dev] = static_cast<unsigned char *>(p);
    }
    *out = g_noalloc_ptr[dev];
    return SW_OK;
}

// The thresholds of build_thresholds (R1, R4, R6), written to caller storage without touching the heap:
// Potts -> out[0]; clock -> out[ci * 2q + cj].
void noalloc_thresholds(int model, int q, double T, uint32_t *out)
{
    if (model == SW_POTTS) {
        out[0] = thr_from_p(1.0 - std::exp(-1.0 / T));
        return;
    }
    const int n = 2 * q;
    const double pi = 3.14159265358979323846;
    double s[2 * SW_MAX_Q];
    for (int k = 0; k < n; ++k) s[k] = (k % q == 0) ? 0.0 : std::sin(pi * (double)k / (double)q);
    for (int a = 0; a < n; ++a)
        for (int b = 0; b < n; ++b) {
            const double pr = s[a] * s[b];
            out[(size_t)a * n + b] = pr > 0.0 ? thr_from_p(1.0 - std::exp(-2.0 * pr / T)) : 0u;
        }
}

// S3 + S4 as sw::k_flip computes them, from `in` to `out` (which may be the same buffer: a thread reads and writes its own site only)
__global__ void k_flip_io(sw::Model md, sw::PhiloxKey key, uint32_t t, const int32_t *__restrict__ labels, const uint8_t *in, uint8_t *out)
{
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= md.N) return;
    const uint32_t r = (uint32_t)labels[i];
    uint32_t w[4];
    sw::philox_stream<sw::STREAM_CLUSTER>(key, r >> 2, t, w);
    const uint32_t ww = (r & 2u) ? ((r & 1u) ? w[3] : w[2]) : ((r & 1u) ? w[1] : w[0]);
    const uint32_t s = in[i];
    uint32_t v = s;
    if (md.model == 0) {
        v = sw::mulhi_q(ww, (uint32_t)md.q);
    } else if (ww >> 31) {
        const uint32_t m = sw::axis_of_sweep(key, t, (uint32_t)md.q);
        v = m + (uint32_t)md.q - s;          // in (0, 2q) for s < q
        if (v >= (uint32_t)md.q) v -= (uint32_t)md.q;
    }
    out[i] = (uint8_t)v;
}

// device memory of device `dev` (cudaPointerGetAttributes allocates nothing)
bool noalloc_on_device(const void *p, int dev)
{
    cudaPointerAttributes a;
    if (cudaPointerGetAttributes(&a, p) != cudaSuccess) { cudaGetLastError(); return false; }
    return (a.type == cudaMemoryTypeDevice && a.device == dev) || a.type == cudaMemoryTypeManaged;
}

}  // namespace

extern "C" int sw_sweep_noalloc(int L, int q, int model, double T, uint64_t seed, uint64_t sweep_index,
                                const uint8_t *d_spins_in, uint8_t *d_spins_out, void *cuda_stream)
{
    if (L > SW_NOALLOC_MAX_L)
        return fail(SW_ERR_UNSUPPORTED, "sw_sweep_noalloc: L = %d exceeds SW_NOALLOC_MAX_L = %d (the static scratch of %zu bytes holds "
                    "5 bytes per site of a %d x %d lattice); use sw_create / sw_create_in for larger lattices",
                    L, SW_NOALLOC_MAX_L, NOALLOC_BYTES, SW_NOALLOC_MAX_L, SW_NOALLOC_MAX_L);
    if (!args_ok(L, q, model) || !(T > 0.0) || !std::isfinite(T))
        return fail(SW_ERR_ARG, "sw_sweep_noalloc: need 2<=L<=%d, 2<=q<=%d, model in {0,1}, finite T>0 (got L=%d q=%d model=%d T=%g)",
                    SW_NOALLOC_MAX_L, SW_MAX_Q, L, q, model, T);
    if (sweep_index > 0xFFFFFFFFull) return fail(SW_ERR_ARG, "sw_sweep_noalloc: sweep index must fit 32 bits");
    if (!d_spins_in || !d_spins_out) return fail(SW_ERR_ARG, "sw_sweep_noalloc: NULL spin buffer");
    const size_t N = (size_t)L * (size_t)L;
    if (d_spins_in != d_spins_out && d_spins_in < d_spins_out + N && d_spins_out < d_spins_in + N)
        return fail(SW_ERR_ARG, "sw_sweep_noalloc: d_spins_in and d_spins_out overlap partially");
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess) {
        cudaGetLastError();
        return fail(SW_ERR_CUDA, "sw_sweep_noalloc: no usable CUDA device (this library has no CPU fallback)");
    }
    if (dev < 0 || dev >= NOALLOC_MAX_DEVICES) return fail(SW_ERR_UNSUPPORTED, "sw_sweep_noalloc: device ordinal %d not below %d", dev, NOALLOC_MAX_DEVICES);
    if (!noalloc_on_device(d_spins_in, dev) || !noalloc_on_device(d_spins_out, dev))
        return fail(SW_ERR_ARG, "sw_sweep_noalloc: d_spins_in / d_spins_out must be device memory of the current device (%d)", dev);
    unsigned char *scratch = nullptr;
    int rc = noalloc_scratch(dev, &scratch);
    if (rc != SW_OK) return rc;

    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    uint32_t *table = reinterpret_cast<uint32_t *>(scratch);
    int32_t *labels = reinterpret_cast<int32_t *>(scratch + NOALLOC_LABELS_OFF);
    uint8_t *bonds = scratch + NOALLOC_BONDS_OFF;

    uint32_t thr[(2 * SW_MAX_Q) * (2 * SW_MAX_Q)];
    noalloc_thresholds(model, q, T, thr);
    sw::Model md{};
    md.L = L; md.q = q; md.model = model; md.N = (uint32_t)N;
    md.thr_potts = model == SW_POTTS ? thr[0] : 0u;
    md.table = table;
    // pageable host memory: the copy is staged before cudaMemcpyAsync returns, so `thr` may leave scope
    if (model == SW_CLOCK) CU_TRY(cudaMemcpyAsync(table, thr, 4 * (size_t)(2 * q) * (2 * q), cudaMemcpyHostToDevice, stream));
    const sw::PhiloxKey key = sw::make_philox_key(seed);
    const uint32_t t = (uint32_t)sweep_index;
    const unsigned bs = 256;
    // every byte of the scratch these kernels read is written here first (labels by k_label_init, bonds by k_bonds,
    // the table by the copy above): whatever the previous call left behind is never seen
    sw::k_bonds<<<blocks_for((N + 1) / 2, bs), bs, 0, stream>>>(md, key, t, d_spins_in, bonds);
    sw::k_label_init<<<blocks_for(N, bs), bs, 0, stream>>>(md.N, labels);
    sw::k_union<<<blocks_for(N, bs), bs, 0, stream>>>(md, bonds, labels);
    sw::k_flatten<<<blocks_for(N, bs), bs, 0, stream>>>(md.N, labels);
    k_flip_io<<<blocks_for(N, bs), bs, 0, stream>>>(md, key, t, labels, d_spins_in, d_spins_out);
    CU_TRY(cudaGetLastError());
    return SW_OK;
}

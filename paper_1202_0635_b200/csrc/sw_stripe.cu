// NEXT-3 of the scope table: ONE lattice sharded over G ranks by row stripes -- "apply the present formulation to
// multi-GPU" is the paper's own outlook; the scheme is SURVEY.md 8(e).
//
// Rank g owns rows [g L / G, (g + 1) L / G).  One sweep t:
//   1. every rank gets the first row of the next stripe (L bytes, periodic)            -> sw_stripe_first_row + exchange
//   2. bonds of its own sites (Philox keyed on GLOBAL site indices: the stripes draw exactly the bonds of the single-GPU
//      run) and labels inside the stripe, +y bonds of its last row left out              -> sw_stripe_label
//   3. every rank publishes, per column, the local root of its first row, the local root of its last row and whether the
//      +y bond of its last row is active (3 L values)                                   -> sw_stripe_export_seam + all-gather
//   4. every rank solves the same tiny union-find over the seam pairs (<= 2 G L nodes; roots by minimum index, so the
//      result is the canonical root of PAPER.md:47)                                     -> sw_seam_solve (host, no device)
//   5. local roots that the seam solve moved are re-pointed; decisions from the CLUSTER stream keyed on the GLOBAL
//      root, spin update                                                                -> sw_stripe_finish
// The result is bit-identical to the single-GPU sweep.  The kernels here are the simple whole-stripe ones (global-memory
// union-find, as the generic back-end); the exchange itself is the caller's (torch.distributed: NCCL between GPUs, gloo
// in the CPU test of the host logic) -- paper_1202_0635_b200/stripes.py.
#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>
#include <unordered_map>
#include <vector>

#include "sw.h"
#include "sw_generic.cuh"
#include "sw_philox.cuh"

namespace swst {

using sw::Model;
using sw::PhiloxKey;

// bonds of the stripe: one thread per pair of sites (2p, 2p + 1) of the stripe; GLOBAL pair index for the BOND stream.
// spins: [rows][L]; halo: the first row of the next stripe (L bytes).
__global__ void k_stripe_bonds(Model md, PhiloxKey key, uint32_t t, uint32_t row0, uint32_t rows, const uint8_t *spins, const uint8_t *halo,
                               uint8_t *bonds)
{
    const uint32_t L = (uint32_t)md.L, n = rows * L;
    const uint32_t p = blockIdx.x * blockDim.x + threadIdx.x;
    if (2u * p >= n) return;
    uint32_t w[4];
    sw::philox_stream<sw::STREAM_BOND>(key, (row0 * L) / 2u + p, t, w);      // L is even: row0 * L is a pair boundary
    const uint32_t q2 = 2u * (uint32_t)md.q;
    uint32_t m = 0u;
    if (md.model == 1) m = sw::axis_of_sweep(key, t, (uint32_t)md.q);
#pragma unroll
    for (int k = 0; k < 2; ++k) {
        const uint32_t i = 2u * p + (uint32_t)k;
        const uint32_t y = i / L, x = i - y * L;
        const uint32_t xr = (x + 1u == L) ? 0u : x + 1u;
        const uint32_t s = spins[i];
        const uint32_t sn[2] = { spins[y * L + xr], (y + 1u == rows) ? halo[x] : spins[(y + 1u) * L + x] };
        uint32_t b = 0u;
#pragma unroll
        for (int d = 0; d < 2; ++d) {
            uint32_t thr;
            if (md.model == 0) thr = (s == sn[d]) ? md.thr_potts : 0u;
            else thr = md.table[sw::clock_c(s, m, q2) * q2 + sw::clock_c(sn[d], m, q2)];
            b |= (w[2 * k + d] < thr) ? (1u << d) : 0u;
        }
        bonds[i] = (uint8_t)b;
    }
}

// union inside the stripe: +x with the periodic wrap, +y only between rows of the stripe (the last row's +y bonds are
// the seam).  Local indices; the root of a piece is its smallest local = smallest global index.
__global__ void k_stripe_union(uint32_t L, uint32_t rows, const uint8_t *bonds, int32_t *labels)
{
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= rows * L) return;
    const uint32_t b = bonds[i];
    if (!b) return;
    const uint32_t y = i / L, x = i - y * L;
    if (b & 1u) sw::uf_union(labels, (int32_t)i, (int32_t)(y * L + ((x + 1u == L) ? 0u : x + 1u)));
    if ((b & 2u) && y + 1u < rows) sw::uf_union(labels, (int32_t)i, (int32_t)((y + 1u) * L + x));
}

// after the flatten: GLOBAL root of every site of the first and of the last row, and the seam bonds of the last row
__global__ void k_stripe_export(uint32_t L, uint32_t rows, uint32_t offset, const int32_t *labels, const uint8_t *bonds, int32_t *first,
                                int32_t *last, uint8_t *seam)
{
    const uint32_t x = blockIdx.x * blockDim.x + threadIdx.x;
    if (x >= L) return;
    first[x] = labels[x] + (int32_t)offset;
    last[x] = labels[(rows - 1u) * L + x] + (int32_t)offset;
    seam[x] = (bonds[(rows - 1u) * L + x] >> 1) & 1u;
}

// roots[k] (GLOBAL index of a local root of this stripe) now belongs to the cluster with canonical root to[k]
__global__ void k_stripe_remap(uint32_t n_map, uint32_t offset, uint32_t n_sites, const int32_t *from, const int32_t *to, int32_t *groot)
{
    const uint32_t k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n_map) return;
    const uint32_t f = (uint32_t)from[k];
    if (f >= offset && f - offset < n_sites) groot[f - offset] = to[k];
}

__global__ void k_stripe_groot_init(uint32_t n, uint32_t offset, const int32_t *labels, int32_t *groot)
{
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n && labels[i] == (int32_t)i) groot[i] = (int32_t)(i + offset);      // a local root is its own global root until remapped
}

// S3 + S4 with the GLOBAL canonical root; final_labels (optional) receives it
__global__ void k_stripe_flip(Model md, PhiloxKey key, uint32_t t, uint32_t n, const int32_t *labels, const int32_t *groot, uint8_t *spins,
                              int32_t *final_labels)
{
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const uint32_t r = (uint32_t)groot[labels[i]];
    if (final_labels) final_labels[i] = (int32_t)r;
    uint32_t w[4];
    sw::philox_stream<sw::STREAM_CLUSTER>(key, r >> 2, t, w);
    const uint32_t ww = (r & 2u) ? ((r & 1u) ? w[3] : w[2]) : ((r & 1u) ? w[1] : w[0]);
    if (md.model == 0) {
        spins[i] = (uint8_t)sw::mulhi_q(ww, (uint32_t)md.q);
    } else if (ww >> 31) {
        const uint32_t m = sw::axis_of_sweep(key, t, (uint32_t)md.q);
        const uint32_t v = m + (uint32_t)md.q - spins[i];
        spins[i] = (uint8_t)(v >= (uint32_t)md.q ? v - (uint32_t)md.q : v);
    }
}

__global__ void k_stripe_init_spins(Model md, PhiloxKey key, uint32_t offset, uint32_t n, uint8_t *spins)
{
    const uint32_t g = blockIdx.x * blockDim.x + threadIdx.x;      // group of 4 sites of the stripe; offset % 4 == 0
    if (4u * g >= n) return;
    uint32_t w[4];
    sw::philox_stream<sw::STREAM_INIT>(key, offset / 4u + g, 0u, w);
#pragma unroll
    for (int k = 0; k < 4; ++k)
        if (4u * g + k < n) spins[4u * g + k] = (uint8_t)sw::mulhi_q(w[k], (uint32_t)md.q);
}

thread_local char g_err[256] = "";

}  // namespace swst

struct sw_stripe {
    int L = 0, q = 0, model = 0, rank = 0, nranks = 1, device = 0;
    uint32_t rows = 0, row0 = 0, n = 0, offset = 0;
    uint64_t t = 0;
    bool labelled = false;
    cudaStream_t stream = nullptr;
    char *ws = nullptr;
    uint8_t *spins = nullptr, *halo = nullptr, *bonds = nullptr, *seam = nullptr;
    int32_t *labels = nullptr, *groot = nullptr, *first = nullptr, *last = nullptr, *map_from = nullptr, *map_to = nullptr, *final_labels = nullptr;
    uint32_t *table = nullptr;
    sw::Model md{};
    sw::PhiloxKey key{};
};

namespace {
inline unsigned nblk(size_t n) { return (unsigned)((n + 255) / 256); }
inline size_t up(size_t x) { return (x + 1023) / 1024 * 1024; }
}  // namespace

extern "C" {

sw_stripe *sw_stripe_create(int L, int q, int model, double T, uint64_t seed, int rank, int nranks)
{
    if (L < 4 || L > SW_MAX_L || q < 2 || q > SW_MAX_Q || (model != SW_POTTS && model != SW_CLOCK) || !(T > 0.0) || !std::isfinite(T) ||
        nranks < 1 || rank < 0 || rank >= nranks || L % nranks != 0 || L % 4 != 0 || L / nranks < 1)
        return nullptr;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) { cudaGetLastError(); return nullptr; }
    sw_stripe *s = new (std::nothrow) sw_stripe();
    if (!s) return nullptr;
    s->L = L; s->q = q; s->model = model; s->rank = rank; s->nranks = nranks;
    s->rows = (uint32_t)(L / nranks); s->row0 = s->rows * (uint32_t)rank; s->n = s->rows * (uint32_t)L; s->offset = s->row0 * (uint32_t)L;
    cudaGetDevice(&s->device);
    const size_t n = s->n, Lz = (size_t)L;
    size_t off = 0;
    const size_t o_spins = off; off += up(n);
    const size_t o_halo = off; off += up(Lz);
    const size_t o_bonds = off; off += up(n);
    const size_t o_seam = off; off += up(Lz);
    const size_t o_lab = off; off += up(4 * n);
    const size_t o_groot = off; off += up(4 * n);
    const size_t o_fin = off; off += up(4 * n);
    const size_t o_first = off; off += up(4 * Lz);
    const size_t o_last = off; off += up(4 * Lz);
    const size_t o_mf = off; off += up(4 * 2 * Lz * (size_t)nranks);
    const size_t o_mt = off; off += up(4 * 2 * Lz * (size_t)nranks);
    const size_t o_tab = off; off += up(4 * (2 * SW_MAX_Q) * (2 * SW_MAX_Q));
    bool ok = cudaMalloc((void **)&s->ws, off) == cudaSuccess && cudaStreamCreateWithFlags(&s->stream, cudaStreamNonBlocking) == cudaSuccess;
    if (!ok) { sw_stripe_destroy(s); return nullptr; }
    s->spins = (uint8_t *)(s->ws + o_spins); s->halo = (uint8_t *)(s->ws + o_halo); s->bonds = (uint8_t *)(s->ws + o_bonds);
    s->seam = (uint8_t *)(s->ws + o_seam); s->labels = (int32_t *)(s->ws + o_lab); s->groot = (int32_t *)(s->ws + o_groot);
    s->final_labels = (int32_t *)(s->ws + o_fin); s->first = (int32_t *)(s->ws + o_first); s->last = (int32_t *)(s->ws + o_last);
    s->map_from = (int32_t *)(s->ws + o_mf); s->map_to = (int32_t *)(s->ws + o_mt); s->table = (uint32_t *)(s->ws + o_tab);
    s->key = sw::make_philox_key(seed);
    // thresholds: DESIGN.md R1 / R4, R6, R7 (host, double, once)
    auto thr = [](double p) -> uint32_t {
        const double v = std::floor(p * 4294967296.0);
        if (!(v > 0.0)) return 0u;
        if (v >= 4294967295.0) return 0xFFFFFFFFu;
        return (uint32_t)v;
    };
    std::vector<uint32_t> tab((size_t)(2 * SW_MAX_Q) * (2 * SW_MAX_Q), 0u);
    s->md.L = L; s->md.q = q; s->md.model = model; s->md.N = (uint32_t)((size_t)L * L); s->md.table = s->table;
    s->md.thr_potts = model == SW_POTTS ? thr(1.0 - std::exp(-1.0 / T)) : 0u;
    if (model == SW_CLOCK) {
        const int nn = 2 * q;
        const double pi = 3.14159265358979323846;
        std::vector<double> sn(nn);
        for (int k = 0; k < nn; ++k) sn[k] = (k % q == 0) ? 0.0 : std::sin(pi * (double)k / (double)q);
        for (int a = 0; a < nn; ++a)
            for (int b = 0; b < nn; ++b)
                if (sn[a] * sn[b] > 0.0) tab[(size_t)a * nn + b] = thr(1.0 - std::exp(-2.0 * sn[a] * sn[b] / T));
    }
    ok = cudaMemcpyAsync(s->table, tab.data(), tab.size() * 4, cudaMemcpyHostToDevice, s->stream) == cudaSuccess;
    if (ok) {
        swst::k_stripe_init_spins<<<nblk((n + 3) / 4), 256, 0, s->stream>>>(s->md, s->key, s->offset, s->n, s->spins);
        ok = cudaGetLastError() == cudaSuccess && cudaStreamSynchronize(s->stream) == cudaSuccess;
    }
    if (!ok) { sw_stripe_destroy(s); return nullptr; }
    return s;
}

void sw_stripe_destroy(sw_stripe *s)
{
    if (!s) return;
    if (s->stream) { cudaStreamSynchronize(s->stream); cudaStreamDestroy(s->stream); }
    if (s->ws) cudaFree(s->ws);
    delete s;
}

int sw_stripe_first_row(sw_stripe *s, uint8_t *host_out)
{
    if (!s || !host_out) return SW_ERR_ARG;
    if (cudaMemcpyAsync(host_out, s->spins, (size_t)s->L, cudaMemcpyDeviceToHost, s->stream) != cudaSuccess ||
        cudaStreamSynchronize(s->stream) != cudaSuccess)
        return SW_ERR_CUDA;
    return SW_OK;
}

int sw_stripe_label(sw_stripe *s, const uint8_t *halo_row_host)
{
    if (!s || !halo_row_host) return SW_ERR_ARG;
    if (s->t > 0xFFFFFFFFull) return SW_ERR_ARG;
    const uint32_t t = (uint32_t)s->t;
    if (cudaMemcpyAsync(s->halo, halo_row_host, (size_t)s->L, cudaMemcpyHostToDevice, s->stream) != cudaSuccess) return SW_ERR_CUDA;
    swst::k_stripe_bonds<<<nblk(s->n / 2), 256, 0, s->stream>>>(s->md, s->key, t, s->row0, s->rows, s->spins, s->halo, s->bonds);
    sw::k_label_init<<<nblk(s->n), 256, 0, s->stream>>>(s->n, s->labels);
    swst::k_stripe_union<<<nblk(s->n), 256, 0, s->stream>>>((uint32_t)s->L, s->rows, s->bonds, s->labels);
    sw::k_flatten<<<nblk(s->n), 256, 0, s->stream>>>(s->n, s->labels);
    swst::k_stripe_groot_init<<<nblk(s->n), 256, 0, s->stream>>>(s->n, s->offset, s->labels, s->groot);
    swst::k_stripe_export<<<nblk((size_t)s->L), 256, 0, s->stream>>>((uint32_t)s->L, s->rows, s->offset, s->labels, s->bonds, s->first, s->last,
                                                                     s->seam);
    if (cudaGetLastError() != cudaSuccess || cudaStreamSynchronize(s->stream) != cudaSuccess) return SW_ERR_CUDA;
    s->labelled = true;
    return SW_OK;
}

int sw_stripe_export_seam(sw_stripe *s, int32_t *first_row_labels, int32_t *last_row_labels, uint8_t *seam_bonds)
{
    if (!s || !first_row_labels || !last_row_labels || !seam_bonds || !s->labelled) return SW_ERR_ARG;
    const size_t Lz = (size_t)s->L;
    if (cudaMemcpyAsync(first_row_labels, s->first, 4 * Lz, cudaMemcpyDeviceToHost, s->stream) != cudaSuccess ||
        cudaMemcpyAsync(last_row_labels, s->last, 4 * Lz, cudaMemcpyDeviceToHost, s->stream) != cudaSuccess ||
        cudaMemcpyAsync(seam_bonds, s->seam, Lz, cudaMemcpyDeviceToHost, s->stream) != cudaSuccess ||
        cudaStreamSynchronize(s->stream) != cudaSuccess)
        return SW_ERR_CUDA;
    return SW_OK;
}

int sw_stripe_finish(sw_stripe *s, int n_map, const int32_t *from, const int32_t *to)
{
    if (!s || n_map < 0 || (n_map > 0 && (!from || !to)) || !s->labelled || n_map > 2 * s->L * s->nranks) return SW_ERR_ARG;
    const uint32_t t = (uint32_t)s->t;
    if (n_map > 0) {
        if (cudaMemcpyAsync(s->map_from, from, 4 * (size_t)n_map, cudaMemcpyHostToDevice, s->stream) != cudaSuccess ||
            cudaMemcpyAsync(s->map_to, to, 4 * (size_t)n_map, cudaMemcpyHostToDevice, s->stream) != cudaSuccess)
            return SW_ERR_CUDA;
        swst::k_stripe_remap<<<nblk((size_t)n_map), 256, 0, s->stream>>>((uint32_t)n_map, s->offset, s->n, s->map_from, s->map_to, s->groot);
    }
    swst::k_stripe_flip<<<nblk(s->n), 256, 0, s->stream>>>(s->md, s->key, t, s->n, s->labels, s->groot, s->spins, s->final_labels);
    if (cudaGetLastError() != cudaSuccess || cudaStreamSynchronize(s->stream) != cudaSuccess) return SW_ERR_CUDA;
    s->labelled = false;
    s->t += 1;
    return SW_OK;
}

int sw_stripe_get_spins(sw_stripe *s, uint8_t *host_out)
{
    if (!s || !host_out) return SW_ERR_ARG;
    if (cudaMemcpyAsync(host_out, s->spins, (size_t)s->n, cudaMemcpyDeviceToHost, s->stream) != cudaSuccess ||
        cudaStreamSynchronize(s->stream) != cudaSuccess)
        return SW_ERR_CUDA;
    return SW_OK;
}

int sw_stripe_get_labels(sw_stripe *s, int32_t *host_out)
{
    if (!s || !host_out || s->t == 0) return SW_ERR_ARG;
    if (cudaMemcpyAsync(host_out, s->final_labels, 4 * (size_t)s->n, cudaMemcpyDeviceToHost, s->stream) != cudaSuccess ||
        cudaStreamSynchronize(s->stream) != cudaSuccess)
        return SW_ERR_CUDA;
    return SW_OK;
}

int sw_stripe_set_spins(sw_stripe *s, const uint8_t *host_in, uint64_t sweep_index)
{
    if (!s || !host_in || sweep_index > 0xFFFFFFFFull) return SW_ERR_ARG;
    for (uint32_t i = 0; i < s->n; ++i)
        if (host_in[i] >= (uint8_t)s->q) return SW_ERR_ARG;
    if (cudaMemcpyAsync(s->spins, host_in, (size_t)s->n, cudaMemcpyHostToDevice, s->stream) != cudaSuccess ||
        cudaStreamSynchronize(s->stream) != cudaSuccess)
        return SW_ERR_CUDA;
    s->t = sweep_index;
    s->labelled = false;
    return SW_OK;
}

uint64_t sw_stripe_sweep_index(sw_stripe *s) { return s ? s->t : 0; }

// Step 4 -- pure host code, no device: every rank runs it on the same gathered arrays and gets the same answer.
// first / last / seam: [G][L] as published by sw_stripe_export_seam of rank g.  The seam below stripe g joins
// last[g][x] with first[(g + 1) % G][x] wherever seam[g][x] != 0.  Output: the local roots whose canonical root
// differs from themselves (from[k] -> to[k], k < *n_map <= 2 G L), sorted by `from`.
int sw_seam_solve(int G, int L, const int32_t *first, const int32_t *last, const uint8_t *seam, int32_t *from, int32_t *to, int *n_map)
{
    if (G < 1 || L < 1 || !first || !last || !seam || !from || !to || !n_map) return SW_ERR_ARG;
    std::unordered_map<int32_t, int32_t> parent;      // node = a local root (global site index); value = its parent
    parent.reserve((size_t)2 * G * L);
    auto find = [&](int32_t a) -> int32_t {
        auto it = parent.find(a);
        if (it == parent.end()) { parent.emplace(a, a); return a; }
        int32_t r = a;
        while (parent[r] != r) r = parent[r];
        while (parent[a] != r) { const int32_t nx = parent[a]; parent[a] = r; a = nx; }     // compress
        return r;
    };
    for (int g = 0; g < G; ++g) {
        const int gn = (g + 1) % G;
        for (int x = 0; x < L; ++x) {
            if (!seam[(size_t)g * L + x]) continue;
            const int32_t ra = find(last[(size_t)g * L + x]), rb = find(first[(size_t)gn * L + x]);
            if (ra == rb) continue;
            if (ra < rb) parent[rb] = ra; else parent[ra] = rb;      // root = smallest index: PAPER.md:47
        }
    }
    std::vector<std::pair<int32_t, int32_t>> out;
    for (auto &kv : parent) {
        const int32_t r = find(kv.first);
        if (r != kv.first) out.emplace_back(kv.first, r);
    }
    std::sort(out.begin(), out.end());
    for (size_t k = 0; k < out.size(); ++k) { from[k] = out[k].first; to[k] = out[k].second; }
    *n_map = (int)out.size();
    return SW_OK;
}

}  // extern "C"

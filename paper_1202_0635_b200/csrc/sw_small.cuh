// Small-lattice back-end (SW_ALGO_SMALL, 2 <= L <= 128) and the small half of the batch path (NEXT-2 of the scope table;
// PAPER.md:83 Table 1 rows L = 256..512 are 2x slower per spin than L >= 2048 on the GTX580 because a small lattice
// cannot fill a GPU, and Figs 3-6, are temperature scans of many small
// lattices).  One CTA owns one lattice: spins, bonds and labels live in shared memory and the CTA runs n sweeps inside
// ONE launch (config 1, L = 64 x 1000 sweeps, is otherwise pure launch latency: SURVEY 7 hard part 5).  A batch of B
// lattices (own temperature and seed each) is a grid of B CTAs.
//
// Per sweep, the same four steps as everywhere, on shared memory:
//   S1 bonds   one Philox call per two sites (R5 BOND stream), threshold compare (R1 / R4, R6)
//   S2 labels  runs of +x bonds by a sequential scan per 16-site segment, then union-find by minimum index with
//              shared-memory atomicMin over the other bonds (the "proper label ... smallest"), then flatten
//   S3 + S4    every site chases to its root, draws the root's word from the CLUSTER stream and takes the decision
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "sw_generic.cuh"
#include "sw_philox.cuh"

namespace sw {

constexpr int SMALL_MAX_L = 128;
constexpr int SMALL_THREADS = 512;
constexpr uint32_t SMALL_SEG = 16u;      // sites per sequential run scan
#ifndef SMALL_JUMP_ROUNDS
#define SMALL_JUMP_ROUNDS 3
#endif
constexpr int SMALL_TABLE_WORDS = (2 * 16) * (2 * 16);

struct SmallLattice {      // per-lattice parameters of a batch (device array, one entry per CTA)
    PhiloxKey key;
    uint32_t thr_potts;
    uint32_t pad;
};

static inline bool small_supported(int L) { return L >= 2 && L <= SMALL_MAX_L; }

// edges that can reach the union-find: every +y bond and the +x bonds at segment ends (rounded up to keep alignment)
__host__ __device__ static inline uint32_t small_edge_cap(uint32_t N) { return (N + N / SMALL_SEG + 2u * SMALL_MAX_L + 15u) / 16u * 16u; }

static inline size_t small_smem_bytes(int L, int model)
{
    const size_t N = (size_t)L * L, Np = (N + 31) / 32 * 32;
    return 4 * Np + Np + Np + 2 * (size_t)small_edge_cap((uint32_t)N) + (model == 1 ? 4 * (size_t)SMALL_TABLE_WORDS : 0);
}

// Label of site i lives in word i ^ ((i >> 5) & 31) of the label array: after the run scan most roots sit at segment
// starts (multiples of 16), which would put them all in banks 0 and 16 (16-way conflicts on every find and atomic); the
// XOR with the 32-block number spreads them over all banks and keeps 32 consecutive sites conflict-free.
__device__ __forceinline__ uint32_t small_slot(uint32_t i) { return i ^ ((i >> 5) & 31u); }

__device__ __forceinline__ uint32_t small_find(volatile uint32_t *lab, uint32_t a, uint32_t &hops)
{
    uint32_t cur = lab[small_slot(a)];
    if (cur != a) {
        uint32_t prev = a, next;
        while (cur > (next = lab[small_slot(cur)])) {
            lab[small_slot(prev)] = next;      // path halving: any ancestor is a valid parent
            prev = cur;
            cur = next;
            ++hops;
        }
    }
    return cur;
}

__device__ __forceinline__ void small_union(uint32_t *lab, uint32_t a, uint32_t b, uint32_t &hops)
{
    for (;;) {
        a = small_find(lab, a, hops);
        b = small_find(lab, b, hops);
        if (a == b) return;
        if (a < b) { const uint32_t tmp = a; a = b; b = tmp; }
        const uint32_t old = atomicMin(lab + small_slot(a), b);   // a > b
        hops += 1u << 16;
        if (old == a) return;
        a = old;
    }
}

// grid = B lattices, block = SMALL_THREADS.  spins: [B][N] (read at the start, written at the end);
// labels_out (optional): [B][N] canonical roots of the LAST sweep of the call; tables: [B][SMALL_TABLE_WORDS] (clock).
template <int MODEL>
__global__ void __launch_bounds__(SMALL_THREADS)
k_small_sweeps(int Li, int qi, const SmallLattice *lats, const uint32_t *tables, uint8_t *spins, int32_t *labels_out, uint32_t t0,
               int n, unsigned long long *stats)
{
    extern __shared__ __align__(16) unsigned char s_raw[];
    const uint32_t L = (uint32_t)Li, q = (uint32_t)qi, N = L * L, Np = (N + 31u) / 32u * 32u;
    uint32_t *lab = reinterpret_cast<uint32_t *>(s_raw);
    uint8_t *sp = s_raw + 4u * Np;
    uint8_t *bd = sp + Np;
    uint16_t *elist = reinterpret_cast<uint16_t *>(bd + Np);                 // union edges: 2 * site + direction
    uint32_t *tab = reinterpret_cast<uint32_t *>(bd + Np + 2u * small_edge_cap(N));
    __shared__ uint32_t s_nedge;
    const uint32_t tid = threadIdx.x, b = blockIdx.x;
    const SmallLattice lt = lats[b];
    const PhiloxKey &key = lt.key;
    uint8_t *g = spins + (size_t)b * N;
    const uint32_t q2 = 2u * q;

    for (uint32_t i = tid; i < N; i += SMALL_THREADS) sp[i] = g[i];
    if (MODEL == 1)
        for (uint32_t k = tid; k < q2 * q2; k += SMALL_THREADS) tab[k] = tables[(size_t)b * SMALL_TABLE_WORDS + k];
    __syncthreads();

    long long ph_t = stats ? clock64() : 0;
#define SW_SMALL_PHASE(i)                                                               \
    if (stats && tid == 0u) {                                                           \
        const long long now_ = clock64();                                               \
        atomicAdd(stats + 8 + (i), (unsigned long long)(now_ - ph_t));                 \
        ph_t = now_;                                                                    \
    }
    for (int it = 0; it < n; ++it) {
        const uint32_t t = t0 + (uint32_t)it;
        uint32_t m = 0u;
        if (MODEL == 1) m = axis_of_sweep(key, t, q);
        // S1: bonds of the site pair (2p, 2p + 1) from one Philox call; every site starts as its own label
        for (uint32_t p = tid; 2u * p < N; p += SMALL_THREADS) {
            uint32_t w[4];
            philox_stream<STREAM_BOND>(key, p, t, w);
#pragma unroll
            for (int k = 0; k < 2; ++k) {
                const uint32_t i = 2u * p + (uint32_t)k;
                if (i >= N) break;
                const uint32_t y = i / L, x = i - y * L;
                const uint32_t xr = (x + 1u == L) ? 0u : x + 1u, yd = (y + 1u == L) ? 0u : y + 1u;
                const uint32_t s = sp[i];
                const uint32_t sn[2] = { sp[y * L + xr], sp[yd * L + x] };
                uint32_t bb = 0u;
#pragma unroll
                for (int d = 0; d < 2; ++d) {
                    uint32_t thr;
                    if (MODEL == 0) thr = (s == sn[d]) ? lt.thr_potts : 0u;
                    else thr = tab[clock_c(s, m, q2) * q2 + clock_c(sn[d], m, q2)];
                    bb |= (w[2 * k + d] < thr) ? (1u << d) : 0u;
                }
                bd[i] = (uint8_t)bb;
            }
        }
        __syncthreads();
        SW_SMALL_PHASE(0)
        // S2a: +x bonds inside a segment of SMALL_SEG sites by a sequential scan (one thread per segment): every site takes
        // the first site of its run as label -- no atomics, trees of depth 1
        {
            const uint32_t segs_per_row = (L + SMALL_SEG - 1u) / SMALL_SEG;
            for (uint32_t sg = tid; sg < L * segs_per_row; sg += SMALL_THREADS) {
                const uint32_t y = sg / segs_per_row, xs = (sg - y * segs_per_row) * SMALL_SEG;
                const uint32_t xe = xs + SMALL_SEG < L ? xs + SMALL_SEG : L;
                uint32_t cur = y * L + xs;
                for (uint32_t x = xs; x < xe; ++x) {
                    const uint32_t i = y * L + x;
                    if (x > xs && !(bd[i - 1u] & 1u)) cur = i;
                    lab[small_slot(i)] = cur;
                }
            }
        }
        __syncthreads();
        SW_SMALL_PHASE(1)
        // S2b: the remaining bonds (+x across a segment end or the periodic seam, every +y that is not parallel to its
        // left neighbour) go to one edge list, compacted with a ballot per warp, ...
        if (tid == 0u) s_nedge = 0u;
        __syncthreads();
        for (uint32_t base = 0u; base < N; base += SMALL_THREADS) {
            const uint32_t i = base + tid;
            bool e1 = false, e2 = false;
            if (i < N) {
                const uint32_t bb = bd[i];
                const uint32_t y = i / L, x = i - y * L;
                e1 = (bb & 1u) && (x + 1u == L || (x + 1u) % SMALL_SEG == 0u);
                // a +y bond whose left neighbour joins the same two runs (both rows linked, both bonds active) is redundant
                e2 = (bb & 2u) && !(x % SMALL_SEG != 0u && (bd[i - 1u] & 3u) == 3u && (bd[((y + 1u == L) ? 0u : y + 1u) * L + x - 1u] & 1u));
            }
            const uint32_t m1 = __ballot_sync(0xFFFFFFFFu, e1), m2 = __ballot_sync(0xFFFFFFFFu, e2);
            const uint32_t lane = tid & 31u, lt_mask = (1u << lane) - 1u;
            uint32_t pos = 0u;
            if (lane == 0u && (m1 | m2)) pos = atomicAdd(&s_nedge, (uint32_t)(__popc(m1) + __popc(m2)));
            pos = __shfl_sync(0xFFFFFFFFu, pos, 0);
            if (e1) elist[pos + (uint32_t)__popc(m1 & lt_mask)] = (uint16_t)(2u * i);
            if (e2) elist[pos + (uint32_t)__popc(m1) + (uint32_t)__popc(m2 & lt_mask)] = (uint16_t)(2u * i + 1u);
        }
        __syncthreads();
        // ... and every thread takes edges from the list: union-find by minimum index, all lanes busy
        uint32_t hops = 0u;
        {
            const uint32_t ne = s_nedge;
            for (uint32_t e = tid; e < ne; e += SMALL_THREADS) {
                const uint32_t code = elist[e], i = code >> 1;
                const uint32_t y = i / L, x = i - y * L;
                const uint32_t j = (code & 1u) ? ((y + 1u == L) ? 0u : y + 1u) * L + x : y * L + ((x + 1u == L) ? 0u : x + 1u);
                small_union(lab, i, j, hops);
            }
        }
        if (stats) { atomicAdd(stats + 4, (unsigned long long)(hops & 0xFFFFu)); atomicAdd(stats + 3, (unsigned long long)(hops >> 16)); }
        __syncthreads();
        SW_SMALL_PHASE(2)
        // S2c: every site points at its root.  The concurrent unions leave chains of about ten links, so first a few
        // rounds of pointer jumping (label <- label of label: plain loads and stores of ancestors, no barrier needed
        // between rounds for correctness, one is kept so that a round sees the previous one), then a read-only chase.
        // Only owners store in this phase, and only ancestors: a chase that races with them still ends at the root.
        {
            volatile uint32_t *vl = lab;
#pragma unroll 1
            for (int round = 0; round < SMALL_JUMP_ROUNDS; ++round) {
                for (uint32_t i = tid; i < N; i += SMALL_THREADS) {
                    const uint32_t p1 = vl[small_slot(i)];
                    const uint32_t p2 = vl[small_slot(p1)];
                    if (p2 != p1) vl[small_slot(i)] = p2;
                }
                __syncthreads();
            }
            for (uint32_t i = tid; i < N; i += SMALL_THREADS) {
                uint32_t r = vl[small_slot(i)], pr;
                while ((pr = vl[small_slot(r)]) != r) r = pr;
                vl[small_slot(i)] = r;
            }
        }
        __syncthreads();
        SW_SMALL_PHASE(3)
        // S3 + S4: decision of the root (CLUSTER stream keyed on the root), new spin.  Nobody reads another site's spin here.
        const bool export_labels = labels_out != nullptr && it == n - 1;
        for (uint32_t i = tid; i < N; i += SMALL_THREADS) {
            const uint32_t r = lab[small_slot(i)];
            if (export_labels) labels_out[(size_t)b * N + i] = (int32_t)r;
            uint32_t w[4];
            philox_stream<STREAM_CLUSTER>(key, r >> 2, t, w);
            const uint32_t ww = (r & 2u) ? ((r & 1u) ? w[3] : w[2]) : ((r & 1u) ? w[1] : w[0]);
            if (MODEL == 0) {
                sp[i] = (uint8_t)mulhi_q(ww, q);
            } else if (ww >> 31) {
                const uint32_t v = m + q - sp[i];          // in (0, 2q)
                sp[i] = (uint8_t)(v >= q ? v - q : v);
            }
        }
        __syncthreads();
        SW_SMALL_PHASE(4)
    }
#undef SW_SMALL_PHASE
    for (uint32_t i = tid; i < N; i += SMALL_THREADS) g[i] = sp[i];
}

static inline cudaError_t small_launch(int model, int B, int L, int q, const SmallLattice *lats, const uint32_t *tables, uint8_t *spins,
                                       int32_t *labels_out, uint32_t t0, int n, cudaStream_t stream, unsigned long long *stats = nullptr)
{
    const size_t smem = small_smem_bytes(L, model);
    static bool attr_set[2] = { false, false };
    if (!attr_set[model != 0]) {
        cudaError_t e = model == 0 ? cudaFuncSetAttribute(k_small_sweeps<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)small_smem_bytes(SMALL_MAX_L, 0))
                                   : cudaFuncSetAttribute(k_small_sweeps<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)small_smem_bytes(SMALL_MAX_L, 1));
        if (e != cudaSuccess) return e;
        attr_set[model != 0] = true;
    }
    if (model == 0) k_small_sweeps<0><<<B, SMALL_THREADS, smem, stream>>>(L, q, lats, tables, spins, labels_out, t0, n, stats);
    else k_small_sweeps<1><<<B, SMALL_THREADS, smem, stream>>>(L, q, lats, tables, spins, labels_out, t0, n, stats);
    return cudaGetLastError();
}

}  // namespace sw

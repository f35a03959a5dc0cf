// Tiled back-end (SW_ALGO_TILED), L % 128 == 0.  One sweep =
//   K1 k_tile_label   S1 + S2a: bonds (Philox, registers) and tile-local labeling of a 128 x 32 tile in shared
//                     memory: horizontal runs by warp ballots, vertical bonds by union-find (atomicMin on the
//                     minimum local index).  Writes tile-local roots (as global site indices) and the bond bits
//                     that cross a tile edge.
//   K2 k_edge_merge   S2b: union of the tile roots across every active cross-tile bond (global atomicMin).
//   K3 k_flip_tiled   S2c + S3 + S4: chase to the global root, decision from the CLUSTER stream, spin update.
// The canonical root is the minimum site index at every level, so the result is the one of the
// generic back-end and of the oracle, bit for bit.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "sw_generic.cuh"
#include "sw_philox.cuh"

namespace sw {

constexpr int TILE_W = 128;  // sites per tile row  = 32 lanes x 4 sites
constexpr int TILE_H = 32;   // rows per tile       = 8 warps x 4 rows
constexpr int TILE_THREADS = 256;
constexpr uint32_t LABEL_MASK = 0x0FFFFFFFu;  // 28 bits of site index (L <= 16384)

struct TiledState {
    uint8_t *hedge = nullptr;  // [L/128][L]  +x bond of the last column of each tile, per lattice row
    uint8_t *vedge = nullptr;  // [L/32][L]   +y bond of the last row of each tile, per lattice column
    int L = 0;
};

static inline bool tiled_supported(int L) { return L >= TILE_W && L % TILE_W == 0 && L % TILE_H == 0; }

static inline size_t tiled_workspace_bytes(int L)
{
    if (!tiled_supported(L)) return 0;
    return (size_t)(L / TILE_W) * L + (size_t)(L / TILE_H) * L + 1024;
}

// ---------------------------------------------------------------------------------------------------------
// shared-memory union-find on local indices (row * 128 + x), minimum index wins
// ---------------------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t sm_find(const volatile uint32_t *lab, uint32_t a)
{
    uint32_t p;
    while ((p = lab[a]) != a) a = p;
    return a;
}

__device__ __forceinline__ void sm_union(uint32_t *lab, uint32_t a, uint32_t b)
{
    for (;;) {
        a = sm_find(lab, a);
        b = sm_find(lab, b);
        if (a == b) return;
        if (a < b) { const uint32_t tmp = a; a = b; b = tmp; }
        const uint32_t old = atomicMin(lab + a, b);
        if (old == a) return;
        a = old;
    }
}

__device__ __forceinline__ uint32_t bytes_eq_mask(uint32_t a, uint32_t b)
{
    // bit k set iff byte k of a equals byte k of b
    const uint32_t x = a ^ b;
    uint32_t m = 0u;
    m |= ((x & 0x000000FFu) == 0u) ? 1u : 0u;
    m |= ((x & 0x0000FF00u) == 0u) ? 2u : 0u;
    m |= ((x & 0x00FF0000u) == 0u) ? 4u : 0u;
    m |= ((x & 0xFF000000u) == 0u) ? 8u : 0u;
    return m;
}

// K1.  grid = (L/128, L/32), block = 256.
__global__ void __launch_bounds__(TILE_THREADS)
k_tile_label(Model md, PhiloxKey key, uint32_t t, const uint8_t *__restrict__ spins, int32_t *__restrict__ labels,
             uint8_t *__restrict__ hedge, uint8_t *__restrict__ vedge)
{
    __shared__ uint32_t lab[TILE_W * TILE_H];
    __shared__ uint32_t s_table[(2 * 16) * (2 * 16)];

    const uint32_t L = (uint32_t)md.L;
    const uint32_t lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
    const uint32_t x0 = blockIdx.x * TILE_W, y0 = blockIdx.y * TILE_H;
    const uint32_t lx = lane * 4u;             // local x of the thread's first site
    const uint32_t gx = x0 + lx;
    const uint32_t q2 = 2u * (uint32_t)md.q;
    uint32_t m = 0u;
    if (md.model == 1) {
        for (uint32_t k = threadIdx.x; k < q2 * q2; k += TILE_THREADS) s_table[k] = md.table[k];
        m = axis_of_sweep(key, t, (uint32_t)md.q);
        __syncthreads();
    }

    // spins of rows 4w .. 4w+4 (the fifth row is the +y neighbour of the fourth), 4 sites per load
    uint32_t srow[5];
#pragma unroll
    for (int r = 0; r < 5; ++r) {
        uint32_t gy = y0 + warp * 4u + r;
        if (gy >= L) gy -= L;
        srow[r] = *reinterpret_cast<const uint32_t *>(spins + (size_t)gy * L + gx);
    }

    uint32_t hbits = 0u, vbits = 0u;  // 4 bits per row, row r at bits [4r, 4r+4)
#pragma unroll
    for (int r = 0; r < 4; ++r) {
        const uint32_t ly = warp * 4u + r;
        const uint32_t gy = y0 + ly;
        // right neighbour of the 4th site: next lane's first byte, or the halo column for lane 31
        uint32_t nxt = __shfl_down_sync(0xFFFFFFFFu, srow[r], 1) & 0xFFu;
        if (lane == 31u) {
            const uint32_t xr = (x0 + TILE_W == L) ? 0u : x0 + TILE_W;
            nxt = spins[(size_t)gy * L + xr];
        }
        const uint32_t right = (srow[r] >> 8) | (nxt << 24);  // byte k = right neighbour of site k
        const uint32_t down = srow[r + 1];
        const uint32_t i0 = gy * L + gx;                       // even, since gx % 4 == 0
        uint32_t wa[4], wb[4];
        philox_stream<STREAM_BOND>(key, i0 >> 1, t, wa);
        philox_stream<STREAM_BOND>(key, (i0 >> 1) + 1u, t, wb);
        uint32_t h, v;
        if (md.model == 0) {
            const uint32_t eh = bytes_eq_mask(srow[r], right), ev = bytes_eq_mask(srow[r], down);
            const uint32_t th = md.thr_potts;
            h = ((wa[0] < th) ? 1u : 0u) | ((wa[2] < th) ? 2u : 0u) | ((wb[0] < th) ? 4u : 0u) | ((wb[2] < th) ? 8u : 0u);
            v = ((wa[1] < th) ? 1u : 0u) | ((wa[3] < th) ? 2u : 0u) | ((wb[1] < th) ? 4u : 0u) | ((wb[3] < th) ? 8u : 0u);
            h &= eh;
            v &= ev;
        } else {
            h = 0u; v = 0u;
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                const uint32_t c = clock_c((srow[r] >> (8 * k)) & 0xFFu, m, q2);
                const uint32_t cr = clock_c((right >> (8 * k)) & 0xFFu, m, q2);
                const uint32_t cd = clock_c((down >> (8 * k)) & 0xFFu, m, q2);
                const uint32_t wh = (k < 2) ? wa[2 * k] : wb[2 * (k - 2)];
                const uint32_t wv = (k < 2) ? wa[2 * k + 1] : wb[2 * (k - 2) + 1];
                h |= (wh < s_table[c * q2 + cr]) ? (1u << k) : 0u;
                v |= (wv < s_table[c * q2 + cd]) ? (1u << k) : 0u;
            }
        }
        // bonds leaving the tile go to the edge arrays and are dropped from the tile-local graph
        if (lane == 31u) {
            hedge[(size_t)blockIdx.x * L + gy] = (uint8_t)((h >> 3) & 1u);
            h &= 7u;
        }
        if (ly == TILE_H - 1) {
            *reinterpret_cast<uint32_t *>(vedge + (size_t)blockIdx.y * L + gx) =
                (v & 1u) | ((v & 2u) << 7) | ((v & 4u) << 14) | ((v & 8u) << 21);
            v = 0u;
        }
        hbits |= h << (4 * r);
        vbits |= v << (4 * r);

        // horizontal runs of this row: label = local index of the run's first site
        const uint32_t s1 = (h & 1u) ? 0u : 1u;
        const uint32_t s2 = (h & 2u) ? s1 : 2u;
        const uint32_t s3 = (h & 4u) ? s2 : 3u;                      // start (within the lane) of site 3's run
        const uint32_t X = __ballot_sync(0xFFFFFFFFu, (h & 8u) != 0u);   // lane j bonded to lane j+1
        const uint32_t Y = __ballot_sync(0xFFFFFFFFu, s3 == 0u);         // lane j fully connected inside
        uint32_t mlane = lane;                                         // lane in which site 0's run starts
        if (lane > 0u && ((X >> (lane - 1u)) & 1u)) {
            const uint32_t Z = X & (Y >> 1);                           // chain continues from lane j+1 into lane j
            const uint32_t W = ~Z & ((1u << (lane - 1u)) - 1u);        // breaks below lane-1
            mlane = W ? (32u - __clz(W)) : 0u;
        }
        const uint32_t s3m = __shfl_sync(0xFFFFFFFFu, s3, mlane);
        const uint32_t rowbase = ly * TILE_W;
        const uint32_t st0 = rowbase + ((mlane == lane) ? lx : (mlane * 4u + s3m));
        uint4 l4;
        l4.x = st0;
        l4.y = s1 ? rowbase + lx + 1u : st0;
        l4.z = s2 ? rowbase + lx + s2 : st0;
        l4.w = s3 ? rowbase + lx + s3 : st0;
        *reinterpret_cast<uint4 *>(lab + rowbase + lx) = l4;
    }
    __syncthreads();

    // vertical bonds: union of the two runs
#pragma unroll
    for (int r = 0; r < 4; ++r) {
        const uint32_t ly = warp * 4u + r;
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            if ((vbits >> (4 * r + k)) & 1u) {
                const uint32_t a = ly * TILE_W + lx + k;
                sm_union(lab, a, a + TILE_W);
            }
        }
    }
    __syncthreads();

    // final find, conversion to global site indices, coalesced 16-byte stores
#pragma unroll
    for (int r = 0; r < 4; ++r) {
        const uint32_t ly = warp * 4u + r;
        const uint4 l4 = *reinterpret_cast<const uint4 *>(lab + ly * TILE_W + lx);
        uint32_t rr[4] = { l4.x, l4.y, l4.z, l4.w };
        int4 out;
        int32_t *o = reinterpret_cast<int32_t *>(&out);
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            const uint32_t root = sm_find(lab, rr[k]);
            o[k] = (int32_t)((y0 + (root >> 7)) * L + x0 + (root & 127u));
        }
        *reinterpret_cast<int4 *>(labels + (size_t)(y0 + ly) * L + gx) = out;
    }
}

// K2.  One thread per tile-edge bond position: first (L/128)*L right-edge bonds, then (L/32)*L bottom-edge bonds.
__global__ void k_edge_merge(Model md, const uint8_t *__restrict__ hedge, const uint8_t *__restrict__ vedge,
                             int32_t *labels, unsigned long long *stats)
{
    const uint32_t L = (uint32_t)md.L;
    const uint32_t nh = (L / TILE_W) * L, nv = (L / TILE_H) * L;
    const uint32_t e = blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= nh + nv) return;
    uint32_t i, j;
    if (e < nh) {
        if (!hedge[e]) return;
        const uint32_t tx = e / L, y = e - tx * L;
        const uint32_t x = tx * TILE_W + TILE_W - 1u;
        const uint32_t xr = (x + 1u == L) ? 0u : x + 1u;
        i = y * L + x;
        j = y * L + xr;
    } else {
        const uint32_t f = e - nh;
        if (!vedge[f]) return;
        const uint32_t ty = f / L, x = f - ty * L;
        const uint32_t y = ty * TILE_H + TILE_H - 1u;
        const uint32_t yd = (y + 1u == L) ? 0u : y + 1u;
        i = y * L + x;
        j = yd * L + x;
    }
    const int32_t a = __ldcg(labels + i), b = __ldcg(labels + j);
    if (stats) atomicAdd(stats + 1, 1ull);
    uf_union(labels, a, b);
}

// K3.  One thread per 4 sites.
__global__ void __launch_bounds__(256)
k_flip_tiled(Model md, PhiloxKey key, uint32_t t, const int32_t *__restrict__ labels, uint8_t *__restrict__ spins)
{
    const uint32_t g = blockIdx.x * blockDim.x + threadIdx.x;
    if (4u * g >= md.N) return;
    const int4 l4 = *reinterpret_cast<const int4 *>(labels + 4u * (size_t)g);
    const int32_t ll[4] = { l4.x, l4.y, l4.z, l4.w };
    uint32_t sp = *reinterpret_cast<const uint32_t *>(spins + 4u * (size_t)g);
    uint32_t m = 0u;
    if (md.model == 1) m = axis_of_sweep(key, t, (uint32_t)md.q);
    uint32_t out = 0u;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const uint32_t r = (uint32_t)uf_find(labels, ll[k]);
        uint32_t w[4];
        philox_stream<STREAM_CLUSTER>(key, r >> 2, t, w);
        const uint32_t ww = (r & 2u) ? ((r & 1u) ? w[3] : w[2]) : ((r & 1u) ? w[1] : w[0]);
        uint32_t s = (sp >> (8 * k)) & 0xFFu;
        if (md.model == 0) {
            s = mulhi_q(ww, (uint32_t)md.q);
        } else if (ww >> 31) {
            const uint32_t v = m + (uint32_t)md.q - s;
            s = v >= (uint32_t)md.q ? v - (uint32_t)md.q : v;
        }
        out |= s << (8 * k);
    }
    *reinterpret_cast<uint32_t *>(spins + 4u * (size_t)g) = out;
}

__global__ void k_resolve_labels(uint32_t N, int32_t *labels)
{
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < N) labels[i] = uf_find(labels, labels[i]);
}

// ---------------------------------------------------------------------------------------------------------
// host side
// ---------------------------------------------------------------------------------------------------------
static inline int tiled_init(TiledState &st, const Model &md, char *ws, uint8_t *, int32_t *, cudaStream_t)
{
    st.L = md.L;
    st.hedge = reinterpret_cast<uint8_t *>(ws);
    st.vedge = st.hedge + (size_t)(md.L / TILE_W) * md.L;
    return 0;
}

static inline void tiled_destroy(TiledState &) {}

constexpr int TILED_NUM_KERNELS = 3;
static const char *const TILED_KERNELS[TILED_NUM_KERNELS] = { "k_tile_label", "k_edge_merge", "k_flip_tiled" };

// ev (optional): ev[0] is recorded before the first kernel, ev[k+1] after kernel k.
static inline int tiled_sweep(TiledState &st, const Model &md, const PhiloxKey &key, uint32_t t, uint8_t *spins,
                              int32_t *labels, cudaStream_t stream, unsigned long long *stats, uint64_t *launches,
                              cudaEvent_t *ev)
{
    const uint32_t L = (uint32_t)md.L;
    dim3 grid(L / TILE_W, L / TILE_H);
    if (ev) cudaEventRecord(ev[0], stream);
    k_tile_label<<<grid, TILE_THREADS, 0, stream>>>(md, key, t, spins, labels, st.hedge, st.vedge);
    if (ev) cudaEventRecord(ev[1], stream);
    const uint32_t ne = (L / TILE_W) * L + (L / TILE_H) * L;
    k_edge_merge<<<(ne + 255) / 256, 256, 0, stream>>>(md, st.hedge, st.vedge, labels, stats);
    if (ev) cudaEventRecord(ev[2], stream);
    k_flip_tiled<<<(md.N / 4 + 255) / 256, 256, 0, stream>>>(md, key, t, labels, spins);
    if (ev) cudaEventRecord(ev[3], stream);
    *launches += 3;
    return cudaPeekAtLastError() == cudaSuccess ? 0 : -1;
}

static inline int tiled_resolve_labels(TiledState &, const Model &md, int32_t *labels, cudaStream_t stream, uint64_t *launches)
{
    k_resolve_labels<<<(md.N + 255) / 256, 256, 0, stream>>>(md.N, labels);
    *launches += 1;
    return cudaPeekAtLastError() == cudaSuccess ? 0 : -1;
}

}  // namespace sw

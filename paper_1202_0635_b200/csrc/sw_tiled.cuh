// Tiled back-end (SW_ALGO_TILED), L % 128 == 0.  One sweep =
//   K0 k_decisions    S3 for every possible root: the "new spin for every label number" of PAPER.md:69 --
//                     one Philox call per 4 consecutive site indices, one byte per site (Potts: new state,
//                     clock: flip bit).  Independent of the configuration.
//   K1 k_strip_label  S1 + S2a.  One warp owns a 128 x 32 tile and walks its rows top to bottom (the raster
//                     order of Hoshen-Kopelman): bonds from Philox in registers; horizontal
//                     runs from warp ballots; every run inherits the smallest label seen through its up-bonds
//                     (segmented min-scan with shuffles) or opens a new label = the index of its first site;
//                     the rare runs that join two labels queue a merge, resolved per tile by atomicMin
//                     union-find on the label array.  Writes provisional labels (site index of the label's
//                     first site) and the bond bits that cross a tile edge.
//   K2 k_edge_merge   S2b: union across every active cross-tile bond (global atomicMin union-find).
//   K3 k_edge_flatten S2c: path compression of the chains that start at tile-edge sites.
//   K4 k_flip_tiled   S4: chase label -> root (short chains), look the root's decision up, update the spin.
// The root of a cluster is its minimum site index at every level, so the result equals the
// generic back-end's and the oracle's bit for bit.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "sw_generic.cuh"
#include "sw_philox.cuh"

namespace sw {

constexpr int TILE_W = 128;  // sites per tile row  = 32 lanes x 4 sites
constexpr int TILE_H = 32;   // rows per tile, walked sequentially by one warp
constexpr int STRIP_WARPS = 4;
constexpr int STRIP_THREADS = 32 * STRIP_WARPS;
constexpr int QCAP = 384;    // merge pairs queued per warp before a flush
constexpr int MAPN = 128;    // entries of the per-warp equivalence map

__device__ __forceinline__ uint32_t map_slot(uint32_t label) { return (label ^ (label >> 7)) & (MAPN - 1); }
constexpr uint32_t NOLABEL = 0xFFFFFFFFu;

struct TiledState {
    uint32_t *hedge = nullptr;   // [L/128][L/32]  bit r = +x bond of the last column of the tile, row 32*ty + r
    uint8_t *vedge = nullptr;    // [L/32][L/4]    4 bits: +y bonds of the last row of the tile, columns 4k..4k+3
    uint8_t *decision = nullptr; // [N]            per-root decision of the current sweep
    int L = 0;
};

static inline bool tiled_supported(int L) { return L >= TILE_W && L % TILE_W == 0 && L % TILE_H == 0; }

static inline size_t tiled_workspace_bytes(int L)
{
    if (!tiled_supported(L)) return 0;
    const size_t N = (size_t)L * L;
    return (size_t)(L / TILE_W) * (L / 32) * 4 + 1024 + (size_t)(L / TILE_H) * (L / 4) + 1024 + N + 1024;
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

// K0.  One thread per 4 consecutive site indices.
__global__ void __launch_bounds__(256)
k_decisions(Model md, PhiloxKey key, uint32_t t, uint8_t *__restrict__ decision)
{
    const uint32_t g = blockIdx.x * blockDim.x + threadIdx.x;
    if (4u * g >= md.N) return;
    uint32_t w[4];
    philox_stream<STREAM_CLUSTER>(key, g, t, w);
    uint32_t out;
    if (md.model == 0) {
        const uint32_t q = (uint32_t)md.q;
        out = mulhi_q(w[0], q) | (mulhi_q(w[1], q) << 8) | (mulhi_q(w[2], q) << 16) | (mulhi_q(w[3], q) << 24);
    } else {
        out = (w[0] >> 31) | ((w[1] >> 31) << 8) | ((w[2] >> 31) << 16) | ((w[3] >> 31) << 24);
    }
    *reinterpret_cast<uint32_t *>(decision + 4u * (size_t)g) = out;
}

// K1.  grid = ceil(tiles / 4), block = 128 (4 warps, one tile each).
__global__ void __launch_bounds__(STRIP_THREADS)
k_strip_label(Model md, PhiloxKey key, uint32_t t, const uint8_t *__restrict__ spins, int32_t *labels,
              uint32_t *__restrict__ hedge, uint8_t *__restrict__ vedge)
{
    __shared__ uint32_t s_table[(2 * 16) * (2 * 16)];
    __shared__ uint2 s_queue[STRIP_WARPS][QCAP];
    __shared__ uint2 s_eqmap[STRIP_WARPS][MAPN];

    const uint32_t L = (uint32_t)md.L;
    const uint32_t lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
    const uint32_t q2 = 2u * (uint32_t)md.q;
    uint32_t m = 0u;
    if (md.model == 1) {
        for (uint32_t k = threadIdx.x; k < q2 * q2; k += STRIP_THREADS) s_table[k] = md.table[k];
        m = axis_of_sweep(key, t, (uint32_t)md.q);
        __syncthreads();
    }
    const uint32_t tiles_x = L / TILE_W;
    const uint32_t tile = blockIdx.x * STRIP_WARPS + warp;
    if (tile >= tiles_x * (L / TILE_H)) return;
    const uint32_t tx = tile % tiles_x, ty = tile / tiles_x;
    const uint32_t x0 = tx * TILE_W, y0 = ty * TILE_H;
    const uint32_t lx = lane * 4u;
    const uint32_t gx = x0 + lx;
    const uint32_t xr = (x0 + TILE_W == L) ? 0u : x0 + TILE_W;   // halo column (periodic)
    const uint32_t lt_mask = (1u << lane) - 1u;
    uint2 *queue = s_queue[warp];
    uint2 *eqmap = s_eqmap[warp];
    uint32_t qn = 0u;                       // queued merge pairs (warp-uniform)
    for (uint32_t k = lane; k < MAPN; k += 32u) eqmap[k] = make_uint2(NOLABEL, NOLABEL);
    __syncwarp();

    // rows are software-pipelined two deep: `cur` = spins of row r, `nxt` = row r+1, `nx2` = row r+2 (in flight);
    // halo bytes (column x0+128, periodic) are carried by lane 31 only
    uint32_t cur = *reinterpret_cast<const uint32_t *>(spins + (size_t)y0 * L + gx);
    uint32_t halo = (lane == 31u) ? spins[(size_t)y0 * L + xr] : 0u;
    uint32_t y1 = y0 + 1u;
    if (y1 == L) y1 = 0u;
    uint32_t nxt = *reinterpret_cast<const uint32_t *>(spins + (size_t)y1 * L + gx);
    uint32_t halo_n = (lane == 31u) ? spins[(size_t)y1 * L + xr] : 0u;
    uint32_t P0 = NOLABEL, P1 = NOLABEL, P2 = NOLABEL, P3 = NOLABEL;   // labels of the row above
    uint32_t up = 0u;                                                  // +y bonds of the row above (4 bits)
    uint32_t hedge_bits = 0u;

#pragma unroll 1
    for (uint32_t r = 0; r < TILE_H; ++r) {
        const uint32_t gy = y0 + r;
        uint32_t gy2 = gy + 2u;
        if (gy2 >= L) gy2 -= L;
        uint32_t nx2 = 0u, halo_2 = 0u;
        if (r + 1u < TILE_H) {   // row r+2 is needed as the +y neighbour of row r+1
            nx2 = *reinterpret_cast<const uint32_t *>(spins + (size_t)gy2 * L + gx);
            if (lane == 31u) halo_2 = spins[(size_t)gy2 * L + xr];
        }

        // ---- S1: bonds of the 4 sites of this lane (2 Philox calls) -------------------------------------
        uint32_t rn = __shfl_down_sync(0xFFFFFFFFu, cur, 1) & 0xFFu;
        if (lane == 31u) rn = halo;
        const uint32_t right = (cur >> 8) | (rn << 24);       // byte k = +x neighbour of site k
        const uint32_t i0 = gy * L + gx;
        uint32_t wa[4], wb[4];
        philox_stream<STREAM_BOND>(key, i0 >> 1, t, wa);
        philox_stream<STREAM_BOND>(key, (i0 >> 1) + 1u, t, wb);
        bool h0, h1, h2, h3, v0, v1, v2, v3;
        if (md.model == 0) {
            const uint32_t th = md.thr_potts;
            const uint32_t dx = cur ^ right, dy = cur ^ nxt;   // byte k zero <=> equal spins
            h0 = wa[0] < th && (dx & 0x000000FFu) == 0u;
            h1 = wa[2] < th && (dx & 0x0000FF00u) == 0u;
            h2 = wb[0] < th && (dx & 0x00FF0000u) == 0u;
            h3 = wb[2] < th && (dx & 0xFF000000u) == 0u;
            v0 = wa[1] < th && (dy & 0x000000FFu) == 0u;
            v1 = wa[3] < th && (dy & 0x0000FF00u) == 0u;
            v2 = wb[1] < th && (dy & 0x00FF0000u) == 0u;
            v3 = wb[3] < th && (dy & 0xFF000000u) == 0u;
        } else {
            uint32_t hh = 0u, vv2 = 0u;
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                const uint32_t c = clock_c((cur >> (8 * k)) & 0xFFu, m, q2);
                const uint32_t cr = clock_c((right >> (8 * k)) & 0xFFu, m, q2);
                const uint32_t cd = clock_c((nxt >> (8 * k)) & 0xFFu, m, q2);
                const uint32_t wh = (k < 2) ? wa[2 * k] : wb[2 * (k - 2)];
                const uint32_t wv = (k < 2) ? wa[2 * k + 1] : wb[2 * (k - 2) + 1];
                hh |= (wh < s_table[c * q2 + cr]) ? (1u << k) : 0u;
                vv2 |= (wv < s_table[c * q2 + cd]) ? (1u << k) : 0u;
            }
            h0 = hh & 1u; h1 = hh & 2u; h2 = hh & 4u; h3 = hh & 8u;
            v0 = vv2 & 1u; v1 = vv2 & 2u; v2 = vv2 & 4u; v3 = vv2 & 8u;
        }
        // bonds that leave the tile are recorded for K2 and dropped from the tile-local graph
        if (lane == 31u) {
            hedge_bits |= (h3 ? 1u : 0u) << r;
            h3 = false;
        }
        uint32_t v = (v0 ? 1u : 0u) | (v1 ? 2u : 0u) | (v2 ? 4u : 0u) | (v3 ? 8u : 0u);
        if (r == TILE_H - 1) {
            vedge[(size_t)ty * (L / 4) + (gx >> 2)] = (uint8_t)v;
            v = 0u;
        }

        // ---- S2a: horizontal runs of this row -----------------------------------------------------------
        const uint32_t s1 = h0 ? 0u : 1u;                       // first site (within the lane) of site k's run
        const uint32_t s2 = h1 ? s1 : 2u;
        const uint32_t s3 = h2 ? s2 : 3u;
        const bool p012 = h0 && h1, p321 = h2 && h1;
        const bool full = p012 && h2;                           // the 4 sites of the lane are one run
        const uint32_t X = __ballot_sync(0xFFFFFFFFu, h3);      // lane j bonded to lane j+1
        const uint32_t Y = __ballot_sync(0xFFFFFFFFu, full);
        const uint32_t C = X & (Y >> 1);                        // run goes on from lane j THROUGH all of lane j+1
        const bool from_left = ((X << 1) >> lane) & 1u;         // lane-1 bonded to this lane
        uint32_t mlane = lane;                                  // lane in which the run of site 0 starts
        if (from_left) {
            const uint32_t W = ~C & (lt_mask >> 1);             // breaks strictly below lane-1
            mlane = W ? (32u - __clz(W)) : 0u;
        }
        const uint32_t s3m = __shfl_sync(0xFFFFFFFFu, s3, mlane);
        const uint32_t rowg = gy * L + x0;                      // global index of the row's first site
        const uint32_t start0 = rowg + ((mlane == lane) ? lx : (mlane * 4u + s3m));

        // ---- labels seen through up-bonds, min per run --------------------------------------------------
        const uint32_t c0 = (up & 1u) ? P0 : NOLABEL, c1 = (up & 2u) ? P1 : NOLABEL;
        const uint32_t c2 = (up & 4u) ? P2 : NOLABEL, c3 = (up & 8u) ? P3 : NOLABEL;
        // head part = sites 0..first break, tail part = sites s3..3
        const uint32_t a = min(min(c0, h0 ? c1 : NOLABEL), min(p012 ? c2 : NOLABEL, full ? c3 : NOLABEL));
        const uint32_t b = min(min(c3, h2 ? c2 : NOLABEL), min(p321 ? c1 : NOLABEL, full ? c0 : NOLABEL));
        // inclusive segmented min-scan of the tail-part values along the run (head lane hl .. this lane)
        const int dist = full ? (int)(lane - mlane) : 0;        // lanes between the run's head lane and this lane
        uint32_t vv = b;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const uint32_t o = __shfl_up_sync(0xFFFFFFFFu, vv, d);
            if (dist >= d) vv = min(vv, o);
        }
        // total of the run that holds this lane's tail part: ends in lane z (tail) or in lane z+1's head part
        const uint32_t z = lane + (uint32_t)__ffs((int)((~C) >> lane)) - 1u;
        uint32_t Tt = __shfl_sync(0xFFFFFFFFu, vv, z);
        const uint32_t ext = __shfl_sync(0xFFFFFFFFu, a, (z + 1u) & 31u);
        if ((X >> z) & 1u) Tt = min(Tt, ext);
        const uint32_t vprev = __shfl_up_sync(0xFFFFFFFFu, vv, 1);
        uint32_t Th = Tt;
        if (!full) Th = from_left ? min(a, vprev) : a;
        const uint32_t mid = min(c1, c2);
        // per-site run minimum
        const uint32_t t1 = h0 ? Th : (p321 ? Tt : (h1 ? mid : c1));
        const uint32_t t2 = h2 ? Tt : (p012 ? Th : (h1 ? mid : c2));
        // a run without any up-bond opens a new label: the global index of its first site
        uint32_t n0 = (Th == NOLABEL) ? start0 : Th;
        uint32_t n1 = (t1 == NOLABEL) ? (s1 ? rowg + lx + 1u : start0) : t1;
        uint32_t n2 = (t2 == NOLABEL) ? (s2 ? rowg + lx + s2 : start0) : t2;
        uint32_t n3 = (Tt == NOLABEL) ? (s3 ? rowg + lx + s3 : start0) : Tt;

        // ---- runs that see two different labels through their up-bonds: the larger label c is merged into the
        // smaller one n.  The pair is queued for the union-find; it is also published in a small direct-mapped
        // map (c -> n) that every lane consults for the labels it hands to the next row, so that merged labels
        // leave the frontier quickly and are not met again and again.  Map entries never go stale: c == n stays
        // a true equivalence.  A collision only loses a shortcut, never a merge.
        const bool m0 = c0 != NOLABEL && c0 != n0, m1 = c1 != NOLABEL && c1 != n1;
        const bool m2 = c2 != NOLABEL && c2 != n2, m3 = c3 != NOLABEL && c3 != n3;
        const uint32_t b0 = __ballot_sync(0xFFFFFFFFu, m0), b1 = __ballot_sync(0xFFFFFFFFu, m1);
        const uint32_t b2 = __ballot_sync(0xFFFFFFFFu, m2), b3 = __ballot_sync(0xFFFFFFFFu, m3);
        if (b0 | b1 | b2 | b3) {
            const uint32_t q0 = qn + __popc(b0 & lt_mask);
            const uint32_t q1 = qn + __popc(b0) + __popc(b1 & lt_mask);
            const uint32_t q2_ = qn + __popc(b0) + __popc(b1) + __popc(b2 & lt_mask);
            const uint32_t q3 = qn + __popc(b0) + __popc(b1) + __popc(b2) + __popc(b3 & lt_mask);
            if (m0) { queue[q0] = make_uint2(c0, n0); eqmap[map_slot(c0)] = make_uint2(c0, n0); }
            if (m1) { queue[q1] = make_uint2(c1, n1); eqmap[map_slot(c1)] = make_uint2(c1, n1); }
            if (m2) { queue[q2_] = make_uint2(c2, n2); eqmap[map_slot(c2)] = make_uint2(c2, n2); }
            if (m3) { queue[q3] = make_uint2(c3, n3); eqmap[map_slot(c3)] = make_uint2(c3, n3); }
            qn += __popc(b0) + __popc(b1) + __popc(b2) + __popc(b3);
            __syncwarp();
        }
        {
            const uint2 e0 = eqmap[map_slot(n0)], e1 = eqmap[map_slot(n1)];
            const uint2 e2 = eqmap[map_slot(n2)], e3 = eqmap[map_slot(n3)];
            n0 = (e0.x == n0) ? e0.y : n0; n1 = (e1.x == n1) ? e1.y : n1;
            n2 = (e2.x == n2) ? e2.y : n2; n3 = (e3.x == n3) ? e3.y : n3;
        }
        *reinterpret_cast<int4 *>(labels + (size_t)gy * L + gx) = make_int4((int)n0, (int)n1, (int)n2, (int)n3);

        if (qn > QCAP - 128 || (r == TILE_H - 1 && qn > 0u)) {   // a row adds at most 128 pairs
            // all label rows written so far must be visible to the atomics of the other lanes
            __threadfence_block();
            __syncwarp();
            for (uint32_t e = lane; e < qn; e += 32u) {
                const uint2 pr = queue[e];
                uf_union(labels, (int32_t)pr.x, (int32_t)pr.y);
            }
            __syncwarp();
            qn = 0u;
        }

        P0 = n0; P1 = n1; P2 = n2; P3 = n3;
        up = v;
        cur = nxt; nxt = nx2;
        halo = halo_n; halo_n = halo_2;
    }
    if (lane == 31u) hedge[(size_t)tx * (L / 32) + ty] = hedge_bits;
}

// Boundary bond e -> (active, owner site i, neighbour site j).  First the (L/128)*L right-edge bonds, then the
// (L/32)*L bottom-edge bonds.
__device__ __forceinline__ bool edge_bond(uint32_t e, uint32_t L, const uint32_t *__restrict__ hedge,
                                          const uint8_t *__restrict__ vedge, uint32_t &i, uint32_t &j)
{
    const uint32_t nh = (L / TILE_W) * L;
    if (e < nh) {
        const uint32_t tx = e / L, y = e - tx * L;
        const uint32_t x = tx * TILE_W + TILE_W - 1u;
        const uint32_t xr = (x + 1u == L) ? 0u : x + 1u;
        i = y * L + x;
        j = y * L + xr;
        return (hedge[tx * (L / 32) + (y >> 5)] >> (y & 31u)) & 1u;
    }
    const uint32_t f = e - nh;
    const uint32_t ty = f / L, x = f - ty * L;
    const uint32_t y = ty * TILE_H + TILE_H - 1u;
    const uint32_t yd = (y + 1u == L) ? 0u : y + 1u;
    i = y * L + x;
    j = yd * L + x;
    return (vedge[ty * (L / 4) + (x >> 2)] >> (x & 3u)) & 1u;
}

// K2.  One thread per tile-edge bond position.
__global__ void __launch_bounds__(256)
k_edge_merge(Model md, const uint32_t *__restrict__ hedge, const uint8_t *__restrict__ vedge, int32_t *labels,
             unsigned long long *stats)
{
    const uint32_t L = (uint32_t)md.L;
    const uint32_t ne = (L / TILE_W) * L + (L / TILE_H) * L;
    const uint32_t e = blockIdx.x * blockDim.x + threadIdx.x;
    uint32_t i = 0u, j = 0u;
    const bool act = (e < ne) && edge_bond(e, L, hedge, vedge, i, j);
    int32_t a = -1, b = -1;
    if (act) { a = __ldcg(labels + i); b = __ldcg(labels + j); }
    // the neighbouring edge position often joins the same pair of labels: skip the repeat
    const int32_t pa = __shfl_up_sync(0xFFFFFFFFu, a, 1), pb = __shfl_up_sync(0xFFFFFFFFu, b, 1);
    const bool dup = (threadIdx.x & 31u) != 0u && pa == a && pb == b;
    if (act && !dup) {
        if (stats) atomicAdd(stats + 1, 1ull);
        uf_union(labels, a, b);
    }
}

// K3.  Path compression from both ends of every active tile-edge bond, so that K4's chases stay short.
__global__ void __launch_bounds__(256)
k_edge_flatten(Model md, const uint32_t *__restrict__ hedge, const uint8_t *__restrict__ vedge, int32_t *labels)
{
    const uint32_t L = (uint32_t)md.L;
    const uint32_t ne = (L / TILE_W) * L + (L / TILE_H) * L;
    const uint32_t e = blockIdx.x * blockDim.x + threadIdx.x;
    uint32_t i = 0u, j = 0u;
    if (e >= ne || !edge_bond(e, L, hedge, vedge, i, j)) return;
    const int32_t a = __ldcg(labels + i), b = __ldcg(labels + j);
    const int32_t root = uf_find(labels, a);     // a and b are in one cluster after K2
    int32_t x = a;
    while (x != root) { const int32_t nx = __ldcg(labels + x); labels[x] = root; x = nx; }
    x = b;
    while (x != root) { const int32_t nx = __ldcg(labels + x); labels[x] = root; x = nx; }
}

// K4.  One thread per 4 sites.
__global__ void __launch_bounds__(256)
k_flip_tiled(Model md, PhiloxKey key, uint32_t t, const int32_t *__restrict__ labels,
             const uint8_t *__restrict__ decision, uint8_t *__restrict__ spins)
{
    const uint32_t g = blockIdx.x * blockDim.x + threadIdx.x;
    if (4u * g >= md.N) return;
    const int4 l4 = *reinterpret_cast<const int4 *>(labels + 4u * (size_t)g);
    int32_t r[4] = { l4.x, l4.y, l4.z, l4.w };
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        int32_t p;
        while ((p = __ldg(labels + r[k])) != r[k]) r[k] = p;
    }
    uint32_t d = 0u;
#pragma unroll
    for (int k = 0; k < 4; ++k) d |= (uint32_t)__ldg(decision + r[k]) << (8 * k);
    if (md.model == 0) {
        *reinterpret_cast<uint32_t *>(spins + 4u * (size_t)g) = d;
    } else if (d) {
        const uint32_t m = axis_of_sweep(key, t, (uint32_t)md.q);
        const uint32_t sp = *reinterpret_cast<const uint32_t *>(spins + 4u * (size_t)g);
        uint32_t out = 0u;
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            uint32_t s = (sp >> (8 * k)) & 0xFFu;
            if ((d >> (8 * k)) & 1u) {
                const uint32_t vv = m + (uint32_t)md.q - s;
                s = vv >= (uint32_t)md.q ? vv - (uint32_t)md.q : vv;
            }
            out |= s << (8 * k);
        }
        *reinterpret_cast<uint32_t *>(spins + 4u * (size_t)g) = out;
    }
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
    const size_t L = (size_t)md.L;
    st.L = md.L;
    st.hedge = reinterpret_cast<uint32_t *>(ws);
    size_t off = ((L / TILE_W) * (L / 32) * 4 + 1023) / 1024 * 1024;
    st.vedge = reinterpret_cast<uint8_t *>(ws + off);
    off += ((L / TILE_H) * (L / 4) + 1023) / 1024 * 1024;
    st.decision = reinterpret_cast<uint8_t *>(ws + off);
    return 0;
}

static inline void tiled_destroy(TiledState &) {}

constexpr int TILED_NUM_KERNELS = 4;
static const char *const TILED_KERNELS[TILED_NUM_KERNELS] = { "k_decisions", "k_strip_label", "k_edge_merge", "k_flip_tiled" };

// ev (optional): ev[0] is recorded before the first kernel, ev[k+1] after kernel k.
static inline int tiled_sweep(TiledState &st, const Model &md, const PhiloxKey &key, uint32_t t, uint8_t *spins,
                              int32_t *labels, cudaStream_t stream, unsigned long long *stats, uint64_t *launches,
                              cudaEvent_t *ev)
{
    const uint32_t L = (uint32_t)md.L;
    const uint32_t tiles = (L / TILE_W) * (L / TILE_H);
    const uint32_t ne = (L / TILE_W) * L + (L / TILE_H) * L;
    if (ev) cudaEventRecord(ev[0], stream);
    k_decisions<<<(md.N / 4 + 255) / 256, 256, 0, stream>>>(md, key, t, st.decision);
    if (ev) cudaEventRecord(ev[1], stream);
    k_strip_label<<<(tiles + STRIP_WARPS - 1) / STRIP_WARPS, STRIP_THREADS, 0, stream>>>(md, key, t, spins, labels, st.hedge,
                                                                                         st.vedge);
    if (ev) cudaEventRecord(ev[2], stream);
    k_edge_merge<<<(ne + 255) / 256, 256, 0, stream>>>(md, st.hedge, st.vedge, labels, stats);
    if (ev) cudaEventRecord(ev[3], stream);
    k_flip_tiled<<<(md.N / 4 + 255) / 256, 256, 0, stream>>>(md, key, t, labels, st.decision, spins);
    if (ev) cudaEventRecord(ev[4], stream);
    *launches += 4;
    return cudaPeekAtLastError() == cudaSuccess ? 0 : -1;
}

static inline int tiled_resolve_labels(TiledState &, const Model &md, int32_t *labels, cudaStream_t stream, uint64_t *launches)
{
    k_resolve_labels<<<(md.N + 255) / 256, 256, 0, stream>>>(md.N, labels);
    *launches += 1;
    return cudaPeekAtLastError() == cudaSuccess ? 0 : -1;
}

}  // namespace sw

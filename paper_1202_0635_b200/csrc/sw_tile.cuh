// Tiled back-end (SW_ALGO_TILED), L % 128 == 0.  One sweep = three kernels, chained by programmatic dependent launch:
//
//   K1 k_tile_label   S1 + S2a + S3 for the clusters that end inside a tile.  One CTA owns a 128 x 64 tile.
//        phase A  bonds: Philox in registers (one call per two sites), compared with the integer threshold; the
//                 2 bits per site are packed into row bit masks H (bond to +x) and V (bond to +y) in shared memory.
//                 Bonds never go to HBM; only the bits that cross a tile edge are exported (hedge / vedge).
//        phase B  labeling on the masks, one thread per 32-site word.  A node = a horizontal run clipped to its
//                 word, named by the tile-local index of its first site, so all +x bonds inside a word are merged by
//                 bit arithmetic alone.  B1: every run with a bond to the row above inherits (plain store) the run
//                 above its lowest such bond; B2: only the remaining, non-redundant up-bonds and the bonds between
//                 words go through the shared-memory union-find (atomicMin, root = smallest index: the "proper
//                 label ... smallest" of PAPER.md:47 at tile level); B3: clusters that may continue in another
//                 tile are marked open by their boundary sites, and the first thread to mark a root registers it as
//                 node tile * OCAP + pos of the global union-find; B3b: the closed roots of all warps are listed
//                 tile-wide and every thread draws one cluster decision per round (CLUSTER stream keyed on the root's
//                 global site index); B4: every run resolves to its root.  Labels in shared memory are entry addresses
//                 (a pointer hop is one LDS), the pointer in the low half of an entry, the output value in the high half.
//        output   one byte per site: decision (closed cluster) or 16 + pos (open cluster) -- the low byte of the 16-bit
//                 value DEC_BASE + decision / LOPEN | 16 + pos that tiles with many open roots write instead; the labels
//                 of the tile's boundary sites also go to a compact edge array for K2.
//   K2 k_seam_merge   S2b: union across every active tile-crossing bond in the global union-find over open roots
//                     (64-bit keys (site index, node), atomicMin: the root of a cluster is its minimum site index).
//   K3 k_tile_flip    S3 for open clusters + S4.  Per tile: one decision per open root, keyed on the site index of its
//                     global root; then every site looks its label up in a 528-byte table and the new spin is
//                     written to the other ping-pong buffer.
//
// The root of a cluster is its minimum site index at both levels (row-major order inside a tile equals the order
// of the global indices), so spins, labels and observables equal the oracle's bit for bit.
// HBM traffic per site and sweep: K1 1 B (spins) + 1 B (labels: 2 B for a tile with more than NARROW_MAX open roots);
// K3 1 B (labels) [+ 1 B spins, clock] + 1 B.
#pragma once
#include <cuda.h>            // CUtensorMap (types only: the encoder is fetched through cudaGetDriverEntryPoint)
#include <cuda_runtime.h>
#include <stdint.h>

#include "sw_generic.cuh"
#include "sw_philox.cuh"

namespace sw {

// ---- TMA (cp.async.bulk.tensor) + mbarrier, raw PTX ---------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long *bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(unsigned long long *bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long *bar, uint32_t parity)
{
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "SW_MBAR_WAIT:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
        "@p bra SW_MBAR_DONE;\n\t"
        "bra SW_MBAR_WAIT;\n\t"
        "SW_MBAR_DONE:\n\t}" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
// one box of a 2D tensor map -> shared memory, completion counted in bytes on the mbarrier
__device__ __forceinline__ void tma_load_2d(void *dst, const CUtensorMap *map, uint32_t x, uint32_t y, unsigned long long *bar)
{
    asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];" ::"r"(
                     smem_u32(dst)),
                 "l"(reinterpret_cast<uint64_t>(map)), "r"(x), "r"(y), "r"(smem_u32(bar))
                 : "memory");
}

// shared-memory atomic add written as PTX (one lane of a warp adds the warp's total)
__device__ __forceinline__ uint32_t atoms_add(uint32_t *p, uint32_t v)
{
    uint32_t old;
    asm volatile("atom.shared.add.u32 %0, [%1], %2;" : "=r"(old) : "r"(smem_u32(p)), "r"(v) : "memory");
    return old;
}

constexpr int TW = 128;                 // sites per tile row = 4 words of 32
constexpr int TH = 64;                  // rows per tile
constexpr int NWORD = TW / 32;
constexpr int TILE_SITES = TW * TH;     // 8192 -> 13-bit local index
constexpr int TILE_THREADS = TH * NWORD;  // one thread per word (256)
constexpr int ROWS_PER_WARP = 8;        // TILE_THREADS / 32 warps x 8 rows = TH
constexpr uint32_t LMASK = 0x3FFFu;     // local index field of a label
constexpr uint32_t LOPEN = 0x8000u;     // cluster may continue in another tile
constexpr int LAB_WORDS = TILE_SITES + TILE_SITES / 32;   // skewed tile-local index sp = p + (p >> 5)
#ifndef SW_EDGE_CAP
#define SW_EDGE_CAP 256   // tests build a variant with tiny lists to drive the overflow paths
#endif
constexpr int EDGE_CAP = SW_EDGE_CAP;           // union edges listed per warp (more are handled by their own thread)
constexpr int NDEC = 16;               // decisions are < q <= 16
constexpr int DEC_BASE = 512;           // lab16 value DEC_BASE + d: "closed cluster, decision d" (= OCAP)
constexpr int ECNT = 2 * TH + 2 * TW;     // edge labels exported per tile: left column, right column, top row, bottom row
constexpr int OCAP = 512;               // open roots listed per tile (<= 128 + 64 + 128 + 64 boundary positions)
// Output value of a site: DEC_BASE + d (closed cluster, decision d < 16) or LOPEN | (POS_BASE + pos) (open cluster, node pos
// of its tile).  POS_BASE = 16 makes the LOW BYTE of the value a complete code whenever the tile has at most NARROW_MAX
// open roots (closed: d < 16, open: 16 + pos <= 255): such a tile ("narrow", almost every tile) writes one byte per site to
// lab8 instead of two to lab16, which halves the label traffic of K1 and K3.  A tile with more open roots, and the label
// export (fuse = 0: the values are 14-bit tile-local indices), use lab16; bit 31 of ocount[tile] says which.
constexpr uint32_t POS_BASE = 16u;
#ifndef SW_NARROW_MAX
#define SW_NARROW_MAX 239   // tests build a variant with a small value to mix both formats
#endif
constexpr uint32_t NARROW_MAX = SW_NARROW_MAX;
constexpr uint32_t WIDE_FLAG = 0x80000000u;
static_assert(NARROW_MAX + POS_BASE <= 255u, "narrow code must fit a byte");
static_assert(2 * (TW + TH) + POS_BASE <= DEC_BASE, "open codes must stay below the closed ones");
static_assert(LAB_WORDS <= (int)LMASK + 1, "skewed local index must fit the label field");
static_assert((TILE_THREADS / 32) * ROWS_PER_WARP == TH, "phase A row split");

// Batches (NEXT-2): the tiles of B lattices of the same L, q, model in one grid.  Global tile g = lattice * tiles per
// lattice + local tile; spins, labels and the seam masks of lattice b sit b strides further; the node, edge and
// open-count arrays are indexed by the global tile, so they need no stride.  Key and thresholds differ per lattice.
struct BatchView {
    uint32_t tiles_per_lattice;
    const PhiloxKey *keys;      // [B]
    const uint32_t *thr;        // [B] Potts threshold
    const uint32_t *tables;     // [B][(2*16)^2] clock tables
};

struct TiledState {
    uint16_t *lab16 = nullptr;   // [L][L] output value of every site of a wide tile (or tile-local root, label export)
    uint8_t *lab8 = nullptr;     // [L][L] low byte of the output value of every site of a narrow tile
    uint32_t *hedge = nullptr;   // [L/128][L/32]  bit (y & 31) of word y >> 5: +x bond of column 128 tx + 127, row y
    uint32_t *vedge = nullptr;   // [L/TH][L/32]   bit (x & 31) of word x >> 5: +y bond of row TH ty + TH - 1, column x
    uint16_t *edges = nullptr;   // [tiles][ECNT]  lab16 values of the tile's boundary sites: left col, right col, top row, bottom row
    uint32_t *ocount = nullptr;  // [tiles]        how many
    int L = 0;
    // TMA: one tensor map per spin buffer of the ping-pong ([L][L] uint8, box = one 128 x 64 tile)
    const uint8_t *map_base[2] = { nullptr, nullptr };
    CUtensorMap map[2];
    // batches: number of lattices in the arrays above, and where their keys / thresholds live
    uint32_t nlat = 1;
    bool batch = false;
    BatchView bv{};
};

static inline bool tiled_supported(int L) { return L >= TW && L % TW == 0 && L % TH == 0; }

static inline size_t tiled_workspace_bytes_n(int L, size_t nlat);
static inline size_t tiled_workspace_bytes(int L) { return tiled_workspace_bytes_n(L, 1); }

// ---- shared-memory union-find by minimum index (same scheme as uf_union in sw_generic.cuh) ------------------
// Labels in shared memory are the 32-bit SHARED-WINDOW ADDRESSES of label entries (base of the label array + 4 x the
// skewed tile-local index; below 2^16): a hop is then one LDS with the pointer as its address, no mask, no shift, no add,
// and the atomics take the address as it is.  The low 16 bits of an entry hold the pointer (the entry's own address for a
// root), the high 16 bits stay 0 until the cluster's output value is known (phases B3, B3b).
__device__ __forceinline__ uint32_t lab_ld(uint32_t a)
{
    uint32_t v;
    asm volatile("ld.volatile.shared.u32 %0, [%1];" : "=r"(v) : "r"(a) : "memory");
    return v;
}
__device__ __forceinline__ uint32_t ptr_ld(uint32_t a)
{
    // the 16-bit pointer field, zero-extended (PTX, so that the compiler keeps plain 32-bit compares on the result)
    uint32_t v;
    asm volatile("ld.volatile.shared.u16 %0, [%1];" : "=r"(v) : "r"(a) : "memory");
    return v;
}
__device__ __forceinline__ void lab_st(uint32_t a, uint32_t v)
{
    asm volatile("st.volatile.shared.u32 [%0], %1;" ::"r"(a), "r"(v) : "memory");
}
__device__ __forceinline__ uint32_t lab_min(uint32_t a, uint32_t v)
{
    uint32_t old;
    asm volatile("atom.shared.min.u32 %0, [%1], %2;" : "=r"(old) : "r"(a), "r"(v) : "memory");
    return old;
}
__device__ __forceinline__ uint32_t lab_or(uint32_t a, uint32_t v)
{
    uint32_t old;
    asm volatile("atom.shared.or.b32 %0, [%1], %2;" : "=r"(old) : "r"(a), "r"(v) : "memory");
    return old;
}

__device__ __forceinline__ uint32_t sfind_halve(uint32_t a)
{
    uint32_t cur = lab_ld(a);
    if (cur != a) {
        uint32_t prev = a, next;
        while (cur > (next = lab_ld(cur))) {
            lab_st(prev, next);
            prev = cur;
            cur = next;
        }
    }
    return cur;
}

__device__ __forceinline__ void sunion(uint32_t a, uint32_t b)
{
    for (;;) {
        a = sfind_halve(a);
        b = sfind_halve(b);
        if (a == b) return;
        if (a < b) { const uint32_t tmp = a; a = b; b = tmp; }
        const uint32_t old = lab_min(a, b);   // a > b
        if (old == a) return;
        a = old;
    }
}

// An A/B switch kept for the record (measured slower on B200): SW_K1_HILO = mask of the Philox
// rounds of the labeling kernel computed as IMAD.HI + IMAD (sw_philox.cuh).
#ifndef SW_K1_HILO
#define SW_K1_HILO 0u
#endif
// position of the highest set bit (x != 0): one FLO (31 - __clz(x) compiles to FLO + a subtraction that is then undone)
__device__ __forceinline__ uint32_t top_bit(uint32_t x)
{
    uint32_t r;
    asm("bfind.u32 %0, %1;" : "=r"(r) : "r"(x));
    return r;
}
__device__ __forceinline__ uint32_t pop_top(uint32_t &c)
{
    // highest bit first: one FLO (bfind); lowest first (__ffs) is BREV + FLO, two trips through the slow XU pipe
    const uint32_t k = top_bit(c);
    c ^= 1u << k;
    return k;
}

// first site (bit position) of the segment that holds bit k; S = mask of segment starts (bit 0 always set)
__device__ __forceinline__ uint32_t seg_start(uint32_t S, uint32_t k) { return top_bit(S & ((2u << k) - 1u)); }

// Global site index of the tile-local root named by label word `v` of a site of the tile with origin (X0, Y0).
__device__ __forceinline__ uint32_t root_site(uint32_t v, uint32_t X0, uint32_t Y0, uint32_t L)
{
    const uint32_t sp = v & LMASK;
    const uint32_t p = sp - sp / 33u;          // undo the skew sp = p + (p >> 5)
    return (Y0 + p / TW) * L + X0 + p % TW;
}

// g = 2 g + [w >= th], th > 0, nth = 2^32 - th: the carry of w + nth shifted into g
__device__ __forceinline__ void ge_shift_in(uint32_t &g, uint32_t w, uint32_t nth)
{
    asm("{\n\t.reg .u32 t;\n\tadd.cc.u32 t, %1, %2;\n\taddc.u32 %0, %0, %0;\n\t}" : "+r"(g) : "r"(w), "r"(nth));
}
// g = 2 g + [w >= th]: the carry flag after w - th (set when there is no borrow) shifted into g
__device__ __forceinline__ void ge_sub_shift_in(uint32_t &g, uint32_t w, uint32_t th)
{
    asm("{\n\t.reg .u32 t;\n\tsub.cc.u32 t, %1, %2;\n\taddc.u32 %0, %0, %0;\n\t}" : "+r"(g) : "r"(w), "r"(th));
}
// Device self-test of the two compare primitives above against the plain comparison (sw_selftest): the clock form
// relies on the carry flag after sub.cc being "no borrow", which is what ptxas emits for sm_100a but not what the PTX
// manual words, so a toolchain that changes it fails this test instead of silently flipping every clock bond.
__global__ void k_selftest_compare(const uint32_t *vals, int n, int *bad)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n * n) return;
    const uint32_t w = vals[i / n], th = vals[i % n];
    const uint32_t ge = w >= th ? 1u : 0u;
    uint32_t g1 = 2u, g2 = 2u;
    ge_sub_shift_in(g2, w, th);
    if (g2 != 4u + ge) atomicAdd(bad, 1);
    if (th != 0u) {                       // the add form is only used with th > 0 (emask covers th == 0)
        ge_shift_in(g1, w, 0u - th);
        if (g1 != 4u + ge) atomicAdd(bad + 1, 1);
    }
}

// K1.  grid = tiles, block = TILE_THREADS.  MODEL 0 = Potts, 1 = clock.
// None of the kernels of the PDL chain qualifies a buffer that another kernel of the chain writes as const __restrict__:
// such loads would compile to ld.global.nc, whose read-only contract does not hold while the producer grid may still be
// draining, and which the "memory" clobber of griddepcontrol.wait does not order (tests/test_abi.py checks the SASS).
#ifndef SW_LABEL_MINB
#define SW_LABEL_MINB 5
#endif
// The 128 x 64 spin bytes of the tile are staged in shared memory by TMA: one cp.async.bulk.tensor box issued by one
// thread, completion on an mbarrier; it lands in the storage of the edge lists, which phase B only starts to use after
// phase A has consumed the spins.  The periodic halo (row below, column to the right: tensor maps do not wrap) comes
// through plain loads issued while the box is in flight.
// BATCH: blockIdx.x is a global tile of a batch (BatchView above); the lattice's Philox key then lives in registers
// instead of the constant bank, which costs the fifth resident CTA.
// STATS: the work counters and per-phase clocks of sw_stats (an instantiation of its own: the production kernel carries
// neither the tests nor the two registers of the phase clock).
template <int MODEL, bool OBS, bool BATCH, bool STATS = false>
__global__ void __launch_bounds__(TILE_THREADS, BATCH ? 4 : SW_LABEL_MINB)
k_tile_label(Model md, PhiloxKey key_one, uint32_t t, const uint8_t *spins, const __grid_constant__ CUtensorMap spin_map,
             uint16_t *lab16, uint8_t *lab8, unsigned long long *parent, uint32_t *hedge, uint32_t *vedge, uint16_t *edges, uint32_t *ocount,
             int fuse, unsigned long long *stats, unsigned long long *obs, BatchView bv)
{
    // OBS (q = 2 Potts only, "+ measurement" of PAPER.md:75): S5 fused into phase A.  With two states the
    // XOR of a spin word with its +x / +y neighbour word has byte 1 exactly on the unequal bonds, so three POPC per four
    // sites (on the otherwise idle XU pipe) give bond_hist[1] and state_hist[1] of S^t; the other two bins follow from
    // the tile's site count.  obs[0..1] += bond_hist, obs[16..17] += state_hist (one row of the record ring).
    __shared__ uint32_t s_obs[2];
    __shared__ uint32_t s_H[TH][NWORD];
    __shared__ uint32_t s_V[TH][NWORD];
    __shared__ uint32_t s_lab[LAB_WORDS];
    __shared__ uint32_t s_nroot, s_nopen;                           // closed roots listed / open roots registered so far
    // s_ew: phase A reads the TMA-staged spins of the tile from it (TILE_SITES bytes), phase B keeps the per-warp edge
    // lists in it ([warp][EDGE_CAP + 1], + dump slot): the two uses never overlap in time
    constexpr int EDGE_WORDS = (TILE_THREADS / 32) * (EDGE_CAP + 1);
    constexpr int EW_WORDS = EDGE_WORDS > TILE_SITES / 4 ? EDGE_WORDS : TILE_SITES / 4;
    __shared__ __align__(128) uint32_t s_ew[EW_WORDS];
    uint32_t(*const s_edge)[EDGE_CAP + 1] = reinterpret_cast<uint32_t(*)[EDGE_CAP + 1]>(s_ew);
    __shared__ uint32_t s_enext[TILE_THREADS / 32];                 // next edge to hand out, per warp
    __shared__ __align__(8) unsigned long long s_bar;               // mbarrier of the staged box
    // clock threshold table (phase A only): it lives in the label array, which nobody touches before phase B -- a table
    // of its own (4 KB) would cost the fifth resident CTA per SM
    uint32_t *const s_table = s_lab;

    if (threadIdx.x == 0u) mbar_init(&s_bar, 1u);
    pdl_prologue();
    const uint32_t L = (uint32_t)md.L;
    const uint32_t tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;
    const uint32_t tiles_x = L / TW;
    const uint32_t lat = BATCH ? blockIdx.x / bv.tiles_per_lattice : 0u;          // lattice of the batch
    const uint32_t ltile = BATCH ? blockIdx.x - lat * bv.tiles_per_lattice : blockIdx.x;
    const uint32_t tx = ltile % tiles_x, ty = ltile / tiles_x;
    const uint32_t x0 = tx * TW, y0 = ty * TH;
    const uint32_t q2 = 2u * (uint32_t)md.q;
    PhiloxKey key_lat;
    if (BATCH) {
        key_lat = bv.keys[lat];
        md.thr_potts = bv.thr[lat];
        md.table = bv.tables + (size_t)lat * (2 * 16) * (2 * 16);
        spins += (size_t)lat * md.N;
        lab16 += (size_t)lat * md.N;
        lab8 += (size_t)lat * md.N;
        hedge += (size_t)lat * tiles_x * (L / 32);
        vedge += (size_t)lat * (L / TH) * (L / 32);
    }
    const PhiloxKey &key = BATCH ? key_lat : key_one;
    // per-phase clocks (lane 0 of every warp), only when the work counters are on: stats[8 + phase]
    long long ph_t = STATS ? clock64() : 0;
    (void)ph_t;
#define SW_PHASE(i)                                                                     \
    if (STATS) {                                                                        \
        const long long now_ = clock64();                                               \
        if (lane == 0u) atomicAdd(stats + 8 + (i), (unsigned long long)(now_ - ph_t)); \
        ph_t = now_;                                                                    \
    }
    // tile-wide list of the closed roots for the balanced decision draw (16-bit entries in s_ew once B2 is done with the edge
    // lists); tests build a variant with a tiny list (SW_RCAP) to drive the overflow path
#ifdef SW_RCAP
    constexpr int RLCAP = SW_RCAP;
#else
    constexpr int RLCAP = 2 * EW_WORDS;
#endif
    static_assert(RLCAP <= 2 * EW_WORDS, "root list must fit the storage of the edge lists");
    uint32_t m = 0u;
    if (tid == 32u) { s_nroot = 0u; s_nopen = 0u; }
    if (OBS && tid < 2u) s_obs[tid] = 0u;
    uint32_t o_neq = 0u, o_one = 0u;
    (void)o_neq; (void)o_one; (void)s_obs;
    if (tid == 0u) {                 // after griddepcontrol.wait: the spins of S^t are complete
        mbar_arrive_expect_tx(&s_bar, (uint32_t)TILE_SITES);
        tma_load_2d(s_ew, &spin_map, x0, (BATCH ? lat * L : 0u) + y0, &s_bar);   // batch map: [B * L][L], lattices stacked
    }
    if (MODEL == 1) {
        for (uint32_t k = tid; k < q2 * q2; k += TILE_THREADS) s_table[k] = md.table[k];
        m = axis_of_sweep(key, t, (uint32_t)md.q);
    }

    // ---------------- phase A: bonds of rows 8 warp .. 8 warp + 7, four sites per lane ----------------------
    {
        const uint32_t gx = x0 + 4u * lane;
        const uint32_t xr = (x0 + TW == L) ? 0u : x0 + TW;   // halo column (periodic)
        const uint32_t ly0 = warp * ROWS_PER_WARP;
        uint32_t row[ROWS_PER_WARP + 1], hal[ROWS_PER_WARP];
        const uint32_t nth = 0u - md.thr_potts;                           // 2^32 - threshold (mod 2^32)
        const uint32_t emask = md.thr_potts ? 0x80808080u : 0u;           // threshold 0: no bond at all
        (void)nth; (void)emask;
        // halo first (plain loads, in flight together with the box): the column right of the tile for lane 31, the row
        // below the tile for the last warp
#pragma unroll
        for (int j = 0; j < ROWS_PER_WARP; ++j) hal[j] = (lane == 31u) ? (uint32_t)spins[(size_t)(y0 + ly0 + j) * L + xr] : 0u;
        row[ROWS_PER_WARP] = 0u;
        if (ly0 + ROWS_PER_WARP == (uint32_t)TH) {
            const uint32_t gy = (y0 + TH == L) ? 0u : y0 + TH;
            row[ROWS_PER_WARP] = *reinterpret_cast<const uint32_t *>(spins + (size_t)gy * L + gx);
        }
        __syncthreads();             // the mbarrier is initialised (thread 0, first statement), s_table / s_obs are written
        mbar_wait(&s_bar, 0u);       // the box has landed
#pragma unroll
        for (int j = 0; j <= ROWS_PER_WARP; ++j) {
            if (ly0 + (uint32_t)j < (uint32_t)TH) row[j] = s_ew[(ly0 + (uint32_t)j) * (TW / 4) + lane];
            if (MODEL == 1) {
                // clock: work on c = (2 s - m) mod 2q from here on (R4), four bytes at a time
                row[j] = clock_c4(row[j], m, q2);
                if (j < ROWS_PER_WARP) hal[j] = clock_c4(hal[j], m, q2) & 0xFFu;
            }
        }
        const uint32_t pair0 = ((y0 + ly0) * L + gx) >> 1;           // (L and gx are multiples of 4)
        const bool writer = (lane & 7u) == 0u;                        // the lane that holds the gathered word of 32 sites
        uint32_t *const hrow = &s_H[ly0][lane >> 3], *const vrow = &s_V[ly0][lane >> 3];
#pragma unroll
        for (int j = 0; j < ROWS_PER_WARP; ++j) {
            const uint32_t cur = row[j], nxt = row[j + 1];
            uint32_t rn = __shfl_down_sync(0xFFFFFFFFu, cur, 1) & 0xFFu;
            if (lane == 31u) rn = hal[j];
            const uint32_t right = (cur >> 8) | (rn << 24);       // byte k = +x neighbour of site k
            const uint32_t c0 = pair0 + (uint32_t)j * (L >> 1);     // counter of the first of this lane's two site pairs in row j
            uint32_t wa[4], wb[4];
            philox_stream<STREAM_BOND, SW_K1_HILO>(key, c0, t, wa);
            philox_stream<STREAM_BOND, SW_K1_HILO>(key, c0 + 1u, t, wb);
            uint32_t hn = 0u, vn = 0u;
            if (MODEL == 0) {
                // [w >= th] is the carry of w + (2^32 - th); add-with-carry shifts it into a nibble (two ALU instructions
                // per bond instead of compare + select + or); equal spins come from a zero-byte test on the XOR.
                const uint32_t dx = cur ^ right, dy = cur ^ nxt;   // byte k zero <=> equal spins (bytes < 16)
                if (OBS) { o_neq += (uint32_t)__popc(dx) + (uint32_t)__popc(dy); o_one += (uint32_t)__popc(cur); }
                const uint32_t zx = ~(dx + 0x7F7F7F7Fu) & emask, zy = ~(dy + 0x7F7F7F7Fu) & emask;
                const uint32_t eqh = (zx * 0x00204081u) >> 28, eqv = (zy * 0x00204081u) >> 28;   // bits 7,15,23,31 -> 0..3
                uint32_t gh = 0u, gv = 0u;
                ge_shift_in(gh, wb[2], nth); ge_shift_in(gh, wb[0], nth); ge_shift_in(gh, wa[2], nth); ge_shift_in(gh, wa[0], nth);
                ge_shift_in(gv, wb[3], nth); ge_shift_in(gv, wb[1], nth); ge_shift_in(gv, wa[3], nth); ge_shift_in(gv, wa[1], nth);
                hn = eqh & ~gh;
                vn = eqv & ~gv;
            } else {
#pragma unroll
                for (int k = 3; k >= 0; --k) {       // highest site first: every bond shifts its bit in from the right
                    const uint32_t c = (cur >> (8 * k)) & 0xFFu, cr = (right >> (8 * k)) & 0xFFu, cd = (nxt >> (8 * k)) & 0xFFu;
                    const uint32_t wh = (k < 2) ? wa[2 * k] : wb[2 * (k - 2)];
                    const uint32_t wv = (k < 2) ? wa[2 * k + 1] : wb[2 * (k - 2) + 1];
                    ge_sub_shift_in(hn, wh, s_table[c * q2 + cr]);
                    ge_sub_shift_in(vn, wv, s_table[c * q2 + cd]);
                }
                hn = ~hn & 0xFu;                      // active <=> word < threshold
                vn = ~vn & 0xFu;
            }
            // gather the nibbles of 8 lanes into one 32-site word: H in the low half, V in the high half
            uint32_t c = hn | (vn << 16);
            c |= __shfl_down_sync(0xFFFFFFFFu, c, 1) << 4;
            c |= __shfl_down_sync(0xFFFFFFFFu, c, 2) << 8;
            const uint32_t c4 = __shfl_down_sync(0xFFFFFFFFu, c, 4);
            if (writer) {
                hrow[j * NWORD] = (c & 0xFFFFu) | (c4 << 16);
                vrow[j * NWORD] = (c >> 16) | (c4 & 0xFFFF0000u);
            }
        }
    }
    if (OBS) {
        o_neq = __reduce_add_sync(0xFFFFFFFFu, o_neq);
        o_one = __reduce_add_sync(0xFFFFFFFFu, o_one);
        if (lane == 0u) { atomicAdd(&s_obs[0], o_neq); atomicAdd(&s_obs[1], o_one); }
    }
    __syncthreads();
    if (OBS && tid < 4u) {
        const uint32_t neq = s_obs[0], one = s_obs[1];
        const uint32_t v = tid == 0u ? 2u * TILE_SITES - neq : tid == 1u ? neq : tid == 2u ? TILE_SITES - one : one;
        atomicAdd(obs + (tid < 2u ? tid : 14u + tid), (unsigned long long)v);
    }

    SW_PHASE(0)
    // bonds that leave the tile: exported for K2, never used by the tile-local graph below
    if (tid < (uint32_t)TH) {
        const uint32_t b = __ballot_sync(0xFFFFFFFFu, (s_H[tid][NWORD - 1] >> 31) & 1u);
        if (lane == 0u) hedge[(size_t)tx * (L / 32) + (y0 >> 5) + warp] = b;
    }
    if (tid < (uint32_t)NWORD) vedge[(size_t)ty * (L / 32) + (x0 >> 5) + tid] = s_V[TH - 1][tid];

    // ---------------- phase B: one thread per word --------------------------------------------------------
    // Label entries are addressed by SKEWED tile-local indices sp = p + (p >> 5) (one pad word per 32-site word), so that
    // the 32 lanes of a warp, which own 32 different words, hit 32 different banks when they touch the same bit position;
    // what is stored and passed around is the shared-window ADDRESS sbase + 4 sp of an entry (see lab_ld above).
    const uint32_t sbase = smem_u32(s_lab);
    constexpr uint32_t OPENBIT = 0x80000000u;                 // entry of a root of an open cluster (= LOPEN of its output value)
    const uint32_t wy = tid / NWORD, ww = tid % NWORD;
    const uint32_t sb = sbase + 132u * tid;                   // address of the entry of the word's first site
    const uint32_t sbu = sb - 528u;                           // ... of the word above (tid - 4)
    const uint32_t h = s_H[wy][ww];
    const uint32_t hin = h & 0x7FFFFFFFu;                     // bonds inside the word
    const uint32_t S = ~(hin << 1);                           // run starts (bit 0 always)
    uint32_t u = 0u, ha = 0u;                                 // bonds to the row above / its in-word bonds
    if (wy > 0u) { u = s_V[wy - 1][ww]; ha = s_H[wy - 1][ww] & 0x7FFFFFFFu; }
    const uint32_t Sa = ~(ha << 1);
    // lowest up-bond of every run, by carry propagation: adding the up-bonds that have a right neighbour in their
    // run (g) to the link mask ripples a carry to the end of the run, where the link bit is 0 and absorbs it.
    const uint32_t g = u & hin, sum = hin + g;
    const uint32_t first = (g & (sum ^ hin)) | (u & ~hin & ~sum);
    // up-bonds that still need a union: not the first of their run, and not parallel to the bond on their left
    // (an up-bond is redundant if a lower up-bond of the same run reaches the same run above: both rows linked all the
    // way between them -- the carry-in mask of C + (u & C), C = links present in both rows)
    const uint32_t C = ha & hin, gC = u & C;
    const uint32_t X = u & ~first & ~((C + gC) ^ C ^ gC);
    const bool hedge_out = (ww + 1u < (uint32_t)NWORD) && (h >> 31);
    uint32_t epos;                                            // this thread's first slot in the warp's edge list
    uint32_t etotal;
    {
        const uint32_t n = __popc(X) + (hedge_out ? 1u : 0u);
        uint32_t incl = n;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const uint32_t o = __shfl_up_sync(0xFFFFFFFFu, incl, d);
            if (lane >= (uint32_t)d) incl += o;
        }
        etotal = __shfl_sync(0xFFFFFFFFu, incl, 31);
        epos = incl - n;
    }
    const uint32_t epos0 = epos;
    if (lane == 0u) s_enext[warp] = 32u;

    SW_PHASE(1)
    // B1: loops over set bits only.  Every run with a bond to the row above inherits (plain store) the run above its
    // lowest up-bond; a run without one becomes its own root; the other up-bonds go to the warp's edge list.
    // cs = start bits of the runs without an up-bond: a carry started at the run start runs along the links of the
    // run while no site has an up-bond and lands on the end bit; the same trick on the reversed word maps end bits
    // to start bits.
    uint32_t cs;
    {
        const uint32_t cend = ((hin & ~u) + (S & ~u)) & ~hin & ~u;
        const uint32_t lr = __brev(hin) >> 1;
        cs = __brev((lr + __brev(cend)) & ~lr);
    }
    {
        uint32_t *el = s_edge[warp];
        for (uint32_t c = cs; c;) {
            const uint32_t k = pop_top(c);
            lab_st(sb + 4u * k, sb + 4u * k);
        }
        // `first` and the start bits of the runs that have an up-bond (S & ~cs) hold one bit per such run, in the same
        // order: both are walked from the top, so the run's start needs no search
        for (uint32_t f = first, fs = S & ~cs; f;) {
            const uint32_t k = top_bit(f), ks = top_bit(fs);
            const uint32_t bit = 1u << k;
            f ^= bit;
            fs ^= 1u << ks;
            lab_st(sb + 4u * ks, sbu + 4u * top_bit(Sa & (2u * bit - 1u)));
        }
        for (uint32_t xr = X; xr;) {
            const uint32_t k = pop_top(xr);
            if (epos < (uint32_t)EDGE_CAP) el[epos] = (sb + 4u * seg_start(S, k)) | ((sbu + 4u * seg_start(Sa, k)) << 16);
            ++epos;
        }
        if (hedge_out) {                                      // bond to the next word of the row
            if (epos < (uint32_t)EDGE_CAP) el[epos] = (sb + 132u) | ((sb + 4u * seg_start(S, 31u)) << 16);
            ++epos;
        }
    }
    __syncthreads();
    SW_PHASE(2)
#ifndef SW_RESOLVE_PASSES
#define SW_RESOLVE_PASSES 2
#endif
#ifndef SW_RESOLVE_HOPS
#define SW_RESOLVE_HOPS 4     // pointer hops per run and pass (3 .. 6 measured: 89.6 / 88.5 / ... us)
#endif

    // B2: the warp's edges, one per lane and round (union-find by minimum index: PAPER.md:47 at tile level)
    {
        const uint32_t ne = etotal < (uint32_t)EDGE_CAP ? etotal : (uint32_t)EDGE_CAP;
        // One edge in flight per lane; a lane that has merged its edge takes the next unclaimed one of the warp's
        // list at once (shared counter), so no lane waits for the slowest edge of a batch.
        {
            uint32_t e = lane, ea = 0u, eb = 0u;
            bool have = e < ne;
            if (have) { const uint32_t v = s_edge[warp][e]; ea = v & 0xFFFFu; eb = v >> 16; }
            while (have) {
                const uint32_t pa = lab_ld(ea), pb = lab_ld(eb);
                const uint32_t ga = lab_ld(pa), gb = lab_ld(pb);
                bool done = false;
                if (pa != ea || pb != eb) {
                    if (ga != pa) lab_st(ea, ga);           // path halving: skip one ancestor on each side
                    if (gb != pb) lab_st(eb, gb);
                    ea = ga; eb = gb;
                } else if (ea == eb) {
                    done = true;
                } else {
                    const uint32_t hi = ea > eb ? ea : eb, lo = ea > eb ? eb : ea;
                    const uint32_t old = lab_min(hi, lo);
                    if (old == hi) done = true;
                    else { ea = old; eb = lo; }                  // hi had a parent already: keep it connected to lo
                }
                if (done) {
                    e = atomicAdd(&s_enext[warp], 1u);
                    have = e < ne;
                    if (have) { const uint32_t v = s_edge[warp][e]; ea = v & 0xFFFFu; eb = v >> 16; }
                }
            }
        }
        if (etotal > (uint32_t)EDGE_CAP) {
            // rare (warp-uniform): the list overflowed; every thread unions its unlisted edges itself.  Everything is
            // computed again from the masks in shared memory, so that the common path keeps no register for this one.
            const uint32_t u2 = wy > 0u ? s_V[wy - 1][ww] : 0u;
            const uint32_t ha2 = wy > 0u ? s_H[wy - 1][ww] & 0x7FFFFFFFu : 0u;
            const uint32_t Sa2 = ~(ha2 << 1);
            const uint32_t g2 = u2 & hin, sum2 = hin + g2;
            const uint32_t first2 = (g2 & (sum2 ^ hin)) | (u2 & ~hin & ~sum2);
            const uint32_t C2 = ha2 & hin, gC2 = u2 & C2;
            uint32_t Xr = u2 & ~first2 & ~((C2 + gC2) ^ C2 ^ gC2);
            const bool hedge2 = (ww + 1u < (uint32_t)NWORD) && (h >> 31);
            const uint32_t n2 = __popc(Xr) + (hedge2 ? 1u : 0u);
            uint32_t incl2 = n2;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
                const uint32_t o = __shfl_up_sync(0xFFFFFFFFu, incl2, d);
                if (lane >= (uint32_t)d) incl2 += o;
            }
            uint32_t slot = incl2 - n2;                         // the slots are taken in the order of B1's loop
            while (Xr) {
                const uint32_t k = pop_top(Xr);
                if (slot >= (uint32_t)EDGE_CAP) sunion(sb + 4u * seg_start(S, k), sbu + 4u * seg_start(Sa2, k));
                ++slot;
            }
            if (hedge2 && slot >= (uint32_t)EDGE_CAP) sunion(sb + 132u, sb + 4u * seg_start(S, 31u));
        }
    }
    __syncthreads();

    SW_PHASE(3)
    // B3: clusters that may continue in another tile: every cluster with a site in the top row or the left column
    // (their bonds belong to the neighbouring tiles), or with an active bond across the right or bottom edge.
    // One boundary site per thread and pass; only the first site of a run (or of a bonded stretch) does the work.
    {
        uint32_t c0 = 0xFFFFFFFFu, c1 = 0xFFFFFFFFu;
        if (tid < (uint32_t)TW) {
            const uint32_t w = tid >> 5, k = tid & 31u;
            const uint32_t S0 = ~((s_H[0][w] & 0x7FFFFFFFu) << 1);
            if ((S0 >> k) & 1u) c0 = sbase + 4u * (33u * w + k);
            const uint32_t hb = s_H[TH - 1][w] & 0x7FFFFFFFu, vb = s_V[TH - 1][w];
            const bool dup = k > 0u && ((vb & hb) >> (k - 1u)) & 1u;
            if (((vb >> k) & 1u) && !dup) c1 = sbase + 4u * (33u * ((TH - 1) * NWORD + w) + seg_start(~(hb << 1), k));
        } else if (tid < (uint32_t)(TW + TH)) {
            c0 = sbase + 4u * (33u * ((tid - TW) * NWORD));
        } else if (tid < (uint32_t)(TW + 2 * TH)) {
            const uint32_t r = tid - (TW + TH);
            const uint32_t hr = s_H[r][NWORD - 1];
            if (hr >> 31) c0 = sbase + 4u * (33u * (r * NWORD + NWORD - 1) + seg_start(~((hr & 0x7FFFFFFFu) << 1), 31u));
        }
#pragma unroll
        for (int c = 0; c < 2; ++c) {
            uint32_t a = c ? c1 : c0;
            if (a != 0xFFFFFFFFu) {
                uint32_t p;
                while ((p = ptr_ld(a)) != a) a = p;
                // The first thread to mark a root registers it: node blockIdx.x * OCAP + pos of the global union-find, its
                // own parent, key = (site, node); the root's entry gets its output value LOPEN | pos in the upper half.
                // (Atomic ORs: other boundary sites of the cluster mark the same entry at the same time.)
                const uint32_t old = lab_or(a, OPENBIT);
                if (!(old & OPENBIT)) {
                    const uint32_t pos = atomicAdd(&s_nopen, 1u);
                    const uint32_t node = blockIdx.x * (uint32_t)OCAP + pos;
                    parent[node] = ((unsigned long long)root_site((a - sbase) >> 2, x0, y0, L) << 32) | node;
                    lab_or(a, (POS_BASE + pos) << 16);
                }
            }
        }
    }
    __syncthreads();

    SW_PHASE(4)
    // B3b: the closed roots of the tile (S3 for the clusters that end inside the tile).  Only a run without a bond to the
    // row above can be a root: every other run was given a smaller parent in B1.  `cand` = start bits of such runs.
    // A closed root's entry gets its final 16-bit output value DEC_BASE + decision in the upper half, drawn from the
    // CLUSTER stream keyed on the root's global site index (R5); the open roots got theirs,
    // LOPEN | pos, in B3.
    uint32_t mine = 0u;                           // this word's closed roots that did not fit
    uint16_t *const rl = reinterpret_cast<uint16_t *>(s_ew);
    {
        uint32_t rall = 0u;                       // this word's closed roots
        uint32_t cand = cs;
        if (MODEL == 1) {
            // A spin on the mirror axis has no active bond at all (its thresholds are 0, R4) and the
            // reflection maps it to itself: a closed singleton whose decision is never used -- no draw.  At most two
            // states lie on the axis (2 s = m mod q); ax = the word's sites in one of them, by zero-byte tests on the
            // word's 32 spins (0x1F: no such state).
            const uint32_t q = (uint32_t)md.q;
            uint32_t a1 = 0x1Fu, a2 = 0x1Fu;
            if ((m & 1u) == 0u) { a1 = m >> 1; if ((q & 1u) == 0u) a2 = (m + q) >> 1; }
            else if (q & 1u) a1 = (m + q) >> 1;
            const uint4 *sp4 = reinterpret_cast<const uint4 *>(spins + (size_t)(y0 + wy) * L + x0 + ww * 32u);
            const uint4 lo = sp4[0], hi = sp4[1];
            const uint32_t wv[8] = { lo.x, lo.y, lo.z, lo.w, hi.x, hi.y, hi.z, hi.w };
            uint32_t ax = 0u;
#pragma unroll
            for (int j = 0; j < 8; ++j) {
                const uint32_t z = (~((wv[j] ^ (a1 * 0x01010101u)) + 0x7F7F7F7Fu) | ~((wv[j] ^ (a2 * 0x01010101u)) + 0x7F7F7F7Fu)) &
                                   0x80808080u;                      // bit 7 of a byte set <=> that spin is on the axis
                ax |= ((z * 0x00204081u) >> 28) << (4 * j);          // bits 7, 15, 23, 31 -> one nibble
            }
            cand &= ~ax;
            while (ax) {                          // (also when B3 marked it open: it has no bond at all, so it is closed)
                const uint32_t k = pop_top(ax);
                lab_st(sb + 4u * k, (sb + 4u * k) | ((fuse ? (uint32_t)DEC_BASE : ((sb - sbase) >> 2) + k) << 16));
            }
        }
        if (wy == 0u) cand = 0u;                  // every cluster with a site in the top row is open
        for (uint32_t c = cand; c;) {
            const uint32_t k = pop_top(c);
            if (lab_ld(sb + 4u * k) == sb + 4u * k) rall |= 1u << k;     // a root, and not open (upper half still 0)
        }
        // The closed roots of all warps go to one tile-wide list (16-bit entries in the storage of the edge lists, which
        // B2 has left), so that after the barrier every thread takes one root per round and all warps carry the same
        // load (the roots of a tile crowd in its upper rows).
        const uint32_t n = (uint32_t)__popc(rall);
        uint32_t incl = n;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const uint32_t o = __shfl_up_sync(0xFFFFFFFFu, incl, d);
            if (lane >= (uint32_t)d) incl += o;
        }
        uint32_t base = 0u;
        if (lane == 31u) base = atoms_add(&s_nroot, incl);
        uint32_t at = __shfl_sync(0xFFFFFFFFu, base, 31) + incl - n;
        for (uint32_t rr = rall; rr;) {
            const uint32_t k = pop_top(rr);
            if (at < (uint32_t)RLCAP) rl[at] = (uint16_t)(sb + 4u * k);
            else mine |= 1u << k;                 // hot configurations: more closed roots than the list holds
            ++at;
        }
    }
    __syncthreads();
    {
        auto decide = [&](uint32_t o) {           // o = address of the entry of a closed root
            const uint32_t sp = (o - sbase) >> 2;
            uint32_t out = sp;
            if (fuse) {
                const uint32_t r = root_site(sp, x0, y0, L);
                uint32_t w[4];
                philox_stream<STREAM_CLUSTER, SW_K1_HILO>(key, r >> 2, t, w);
                const uint32_t wsel = (r & 2u) ? ((r & 1u) ? w[3] : w[2]) : ((r & 1u) ? w[1] : w[0]);
                out = (uint32_t)DEC_BASE + (MODEL == 0 ? mulhi_q(wsel, (uint32_t)md.q) : (wsel >> 31));
            }
            lab_st(o, o | (out << 16));
        };
        const uint32_t nc0 = s_nroot, nc = nc0 < (uint32_t)RLCAP ? nc0 : (uint32_t)RLCAP;
        for (uint32_t i = tid; i < nc; i += TILE_THREADS) decide(rl[i]);
        while (mine) {
            const uint32_t k = pop_top(mine);
            decide(sb + 4u * k);
        }
    }
    __syncthreads();

    SW_PHASE(7)
    // B4a: resolve every run of the word to its root's entry (whose upper half is the output value).  Two runs at
    // a time, SW_RESOLVE_HOPS pointer hops each (the loads of one level are independent, so their latencies overlap; all but
    // the last read the 16-bit pointer only), result written back to the run's own entry; runs deeper than that (rare) are
    // finished by a chase that starts from the already advanced pointer.
    uint32_t hops = 0u;
    {
        // one pass over the runs in `todo`: returns the runs that are still not at their root
        auto pass = [&](uint32_t todo) -> uint32_t {
            uint32_t rem = 0u;
            while (todo) {
                // the lowest and the highest run still to do (the same run when one is left: harmless repeat)
                const uint32_t k0 = (uint32_t)__ffs((int)todo) - 1u, k1 = top_bit(todo);
                todo &= todo - 1u;
                todo &= ~(1u << k1);
                uint32_t x0 = ptr_ld(sb + 4u * k0), x1 = ptr_ld(sb + 4u * k1);
                x0 = ptr_ld(x0); x1 = ptr_ld(x1);
#pragma unroll
                for (int hh = 0; hh < SW_RESOLVE_HOPS - 3; ++hh) { x0 = ptr_ld(x0); x1 = ptr_ld(x1); }
                const uint32_t y0r = lab_ld(x0), y1r = lab_ld(x1);
                lab_st(sb + 4u * k0, y0r);
                lab_st(sb + 4u * k1, y1r);
                if ((y0r ^ x0) & 0xFFFCu) rem |= 1u << k0;         // pointer fields differ (offsets are multiples of 4)
                if ((y1r ^ x1) & 0xFFFCu) rem |= 1u << k1;
            }
            return rem;
        };
        uint32_t rem = pass(S);
#pragma unroll 1
        for (int r = 0; r < SW_RESOLVE_PASSES - 1; ++r) rem = pass(rem);   // the written-back pointers of all runs shorten these
        while (rem) {
            const uint32_t k = top_bit(rem);
            rem ^= 1u << k;
            uint32_t a = ptr_ld(sb + 4u * k), p;
            while ((p = ptr_ld(a)) != a) { a = p; ++hops; }
            lab_st(sb + 4u * k, lab_ld(a));
        }
    }
    __syncwarp();
    SW_PHASE(5)

    // B4b: per-site labels of the word: 32 contiguous bytes (narrow tile) or 64 (wide tile, label export)
    {
        const uint32_t nopen = s_nopen;
        const bool narrow = fuse && nopen <= NARROW_MAX;
        if (tid == 0u) ocount[blockIdx.x] = nopen | (narrow ? 0u : WIDE_FLAG);
        uint32_t xs[32];
        uint32_t sbr = sb;                        // pinned in a register: else the address is rebuilt for every predicated load
        asm volatile("" : "+r"(sbr));
#pragma unroll
        for (int k = 0; k < 32; ++k) xs[k] = ((S >> k) & 1u) ? lab_ld(sbr + 4u * k) : 0u;
        uint16_t *ed = edges + (size_t)blockIdx.x * ECNT;       // the labels of the tile's boundary sites, compact, for K2
        const bool edge_row = wy == 0u || wy == (uint32_t)TH - 1u;
        uint32_t cur = 0u;
        if (narrow) {
            uint32_t o8[8];
#pragma unroll
            for (int k = 0; k < 32; ++k) {
                if ((S >> k) & 1u) cur = xs[k];      // upper half = output value of the run's root (B3, B3b); byte 2 = its low byte
                o8[k >> 2] = (k & 3) == 0 ? (cur >> 16) & 0xFFu : __byte_perm(o8[k >> 2], cur, (k & 3) == 1 ? 0x3260 : (k & 3) == 2 ? 0x3610 : 0x6210);
            }
            uint4 *dst = reinterpret_cast<uint4 *>(lab8 + (size_t)(y0 + wy) * L + x0 + ww * 32u);
            dst[0] = make_uint4(o8[0], o8[1], o8[2], o8[3]);
            dst[1] = make_uint4(o8[4], o8[5], o8[6], o8[7]);
            if (edge_row) {                          // K2 reads 16-bit entries: the bytes, zero-extended (it uses the low 10 bits)
                uint4 *de = reinterpret_cast<uint4 *>(ed + 2 * TH + (wy ? TW : 0) + ww * 32u);
#pragma unroll
                for (int c = 0; c < 4; ++c)
                    de[c] = make_uint4(__byte_perm(o8[2 * c], 0u, 0x4140), __byte_perm(o8[2 * c], 0u, 0x4342),
                                       __byte_perm(o8[2 * c + 1], 0u, 0x4140), __byte_perm(o8[2 * c + 1], 0u, 0x4342));
            }
        } else {
            uint32_t o[16];
#pragma unroll
            for (int k = 0; k < 32; ++k) {
                if ((S >> k) & 1u) cur = xs[k];
                if (k & 1) o[k >> 1] |= cur & 0xFFFF0000u; else o[k >> 1] = cur >> 16;
            }
            uint4 *dst = reinterpret_cast<uint4 *>(lab16 + (size_t)(y0 + wy) * L + x0 + ww * 32u);
#pragma unroll
            for (int c = 0; c < 4; ++c) dst[c] = make_uint4(o[4 * c], o[4 * c + 1], o[4 * c + 2], o[4 * c + 3]);
            if (edge_row) {
                uint4 *de = reinterpret_cast<uint4 *>(ed + 2 * TH + (wy ? TW : 0) + ww * 32u);
#pragma unroll
                for (int c = 0; c < 4; ++c) de[c] = make_uint4(o[4 * c], o[4 * c + 1], o[4 * c + 2], o[4 * c + 3]);
            }
        }
        // left / right column: the first and the last run's value (bit 0 of S is always set); a narrow tile exports the
        // low byte only, like its rows
        const uint32_t emask = narrow ? 0xFFu : 0xFFFFu;
        if (ww == 0u) ed[wy] = (uint16_t)((xs[0] >> 16) & emask);
        if (ww == (uint32_t)NWORD - 1u) ed[TH + wy] = (uint16_t)((cur >> 16) & emask);
        SW_PHASE(6)
        if (STATS) {
            const uint32_t n2 = __reduce_add_sync(0xFFFFFFFFu, (uint32_t)__popc(S));
            const uint32_t n3 = __reduce_add_sync(0xFFFFFFFFu, epos - epos0);
            const uint32_t n4 = __reduce_add_sync(0xFFFFFFFFu, hops);
            if (lane == 0u) {
                atomicAdd(stats + 2, (unsigned long long)n2);
                atomicAdd(stats + 3, (unsigned long long)n3);
                atomicAdd(stats + 4, (unsigned long long)n4);
            }
        }
    }
}

// ---- global union-find over the open roots ------------------------------------------------------------------------
// Node n = tile * OCAP + pos.  parent[n] = key of n's parent, key(m) = (site index of m) << 32 | m; a root holds its own
// key.  Keys order the nodes by site index, so hooking the larger root under the smaller one (64-bit atomicMin) makes the
// root of every cluster its minimum site index: the "proper label ... smallest" of PAPER.md:47.  Parents only ever
// decrease, so a stale read is still an ancestor and the atomicMin re-validates the root.
__device__ __forceinline__ unsigned long long gfind(unsigned long long *parent, uint32_t x)
{
    // plain (L1-cacheable) loads: a stale line still holds an ancestor, and hot roots stay out of L2
    unsigned long long p = parent[x];
    uint32_t prev = x;
    while ((uint32_t)p != prev) {
        const uint32_t cur = (uint32_t)p;
        const unsigned long long g = parent[cur];
        if ((uint32_t)g == cur) return g;
        parent[prev] = g;                     // path halving
        prev = cur;
        p = g;
    }
    return p;
}

__device__ __forceinline__ void gunion(unsigned long long *parent, uint32_t x, uint32_t y)
{
    for (;;) {
        unsigned long long kx = gfind(parent, x), ky = gfind(parent, y);
        if (kx == ky) return;
        if (kx < ky) { const unsigned long long tmp = kx; kx = ky; ky = tmp; }
        const unsigned long long old = atomicMin(parent + (uint32_t)kx, ky);   // kx > ky
        if (old == kx) return;                // kx was a root and now hangs under ky
        x = (uint32_t)old;                    // kx already had a parent: keep that parent connected to ky
        y = (uint32_t)ky;
    }
}

// read-only find (K3, label export): site index of the root of node x
__device__ __forceinline__ uint32_t groot_site(const unsigned long long *parent, uint32_t x)
{
    unsigned long long p = __ldcg(parent + x);
    while ((uint32_t)p != x) { x = (uint32_t)p; p = __ldcg(parent + x); }
    return (uint32_t)(p >> 32);
}

// find with write-back (K3): the node itself is re-pointed to the root, so chases of other tiles that pass through it
// end one hop later.  A racing reader sees the old parent or the root: both are ancestors.
__device__ __forceinline__ uint32_t groot_site_compress(unsigned long long *parent, uint32_t x)
{
    const uint32_t x0 = x;
    unsigned long long p = __ldcg(parent + x);
    uint32_t hops = 0u;
    while ((uint32_t)p != x) { x = (uint32_t)p; p = __ldcg(parent + x); ++hops; }
    if (hops > 1u) __stcg(parent + x0, p);
    return (uint32_t)(p >> 32);
}

// K2.  One thread per tile-edge bond position: first the (L/128)*L right-edge bonds, then the (L/TH)*L bottom-edge
// bonds.  The two ends of an active tile-crossing bond lie in open clusters; their lab16 values (LOPEN | pos) come
// from the compact edge arrays K1 wrote.
constexpr int SEAM_THREADS = 256;
// nlat lattices (1 unless a batch): positions of lattice b are b * ne .. (b + 1) * ne - 1, its tiles b * tiles .. .
__global__ void __launch_bounds__(SEAM_THREADS)
k_seam_merge(Model md, const uint32_t *hedge, const uint32_t *vedge, const uint16_t *edges, unsigned long long *parent,
             unsigned long long *stats, uint32_t nlat)
{
    const uint32_t L = (uint32_t)md.L;
    const uint32_t tiles_x = L / TW, tiles_y = L / TH;
    const uint32_t nh = tiles_x * L, ne = nh + tiles_y * L;
    // blocks take the positions in reverse order (bottom edges of the lowest tiles first): measured 0.5-1 us faster per
    // sweep than the forward order at L=4096 (the union order shapes the chains that K2 and K3 have to walk)
    uint32_t e = (gridDim.x - 1u - blockIdx.x) * blockDim.x + threadIdx.x;
    pdl_prologue();
    if (e >= ne * nlat) return;
    const uint32_t lat = e / ne;          // ne is a multiple of 32: uniform in a warp
    e -= lat * ne;
    hedge += (size_t)lat * tiles_x * (L / 32);
    vedge += (size_t)lat * tiles_y * (L / 32);
    const uint32_t tbase = lat * tiles_x * tiles_y;      // node keys carry GLOBAL node numbers: tiles stay global
    uint32_t bit, ta, tb, ia, ib;
    if (e < nh) {
        const uint32_t tx = e / L, y = e - tx * L;
        bit = (hedge[tx * (L / 32) + (y >> 5)] >> (y & 31u)) & 1u;
        ta = tbase + (y / TH) * tiles_x + tx;
        tb = tbase + (y / TH) * tiles_x + (tx + 1u == tiles_x ? 0u : tx + 1u);
        ia = TH + y % TH;                     // right column of ta
        ib = y % TH;                          // left column of tb
    } else {
        const uint32_t f = e - nh;
        const uint32_t ty = f / L, x = f - ty * L;
        bit = (vedge[ty * (L / 32) + (x >> 5)] >> (x & 31u)) & 1u;
        ta = tbase + ty * tiles_x + x / TW;
        tb = tbase + (ty + 1u == tiles_y ? 0u : ty + 1u) * tiles_x + x / TW;
        ia = 2 * TH + TW + x % TW;            // bottom row of ta
        ib = 2 * TH + x % TW;                 // top row of tb
    }
    const uint32_t a = edges[(size_t)ta * ECNT + ia], b = edges[(size_t)tb * ECNT + ib];
    const uint32_t act = __ballot_sync(0xFFFFFFFFu, bit != 0u);   // ne is a multiple of 32: whole warps get here
    if (!bit) return;
    // The 32 positions of a warp lie on one seam of one pair of tiles (32 | TH, 32 | TW), and neighbouring bonds mostly
    // join the same two clusters: one lane per distinct (a, b) pair does the union (SURVEY 7 hard part 3).
    const uint32_t pair = (a << 16) | (b & 0xFFFFu);
    const uint32_t same = __match_any_sync(act, pair);
    if ((uint32_t)__ffs((int)same) - 1u != (threadIdx.x & 31u)) return;
    if (stats) atomicAdd(stats + 1, 1ull);
    gunion(parent, ta * OCAP + ((a & 0x3FFu) - POS_BASE), tb * OCAP + ((b & 0x3FFu) - POS_BASE));
}

// K3.  grid = tiles, block = TILE_THREADS; 32 sites per thread (4 passes of 8).  in = S^t, out = S^{t+1}.
// Resident CTAs per SM: 8 (all 2048 threads) for the Potts kernel -- no difference while the labels sit in L2 (L <= 4096), but
// beyond that the kernel streams from HBM and every tile first waits for the chase of its open roots: 183 -> 140 us at
// L = 16384; the clock kernel keeps more registers (old spins in flight) and stops at 6.
#ifndef SW_FLIP_MINB
#define SW_FLIP_MINB(MODEL, BATCH) ((BATCH) ? 4 : (MODEL) == 0 ? 8 : 6)
#endif
template <int MODEL, bool BATCH>
__global__ void __launch_bounds__(TILE_THREADS, SW_FLIP_MINB(MODEL, BATCH))
k_tile_flip(Model md, PhiloxKey key_one, uint32_t t, const uint16_t *lab16, const uint8_t *lab8, unsigned long long *parent, const uint32_t *ocount,
            const uint8_t *in, uint8_t *out, BatchView bv)
{
    constexpr int PASSES = TILE_SITES / 8 / TILE_THREADS;   // 4
    // decision table, indexed by the low 10 bits of a site's output value (wide tile) or by its low byte (narrow tile):
    // [d] = [DEC_BASE + d] = d for the closed clusters, [POS_BASE + pos] = decision of the tile's open root pos
    __shared__ uint8_t s_dec[DEC_BASE + NDEC];

    const uint32_t L = (uint32_t)md.L;
    const uint32_t tid = threadIdx.x;
    const uint32_t tiles_x = L / TW;
    const uint32_t lat = BATCH ? blockIdx.x / bv.tiles_per_lattice : 0u;
    const uint32_t ltile = BATCH ? blockIdx.x - lat * bv.tiles_per_lattice : blockIdx.x;
    const uint32_t tx = ltile % tiles_x, ty = ltile / tiles_x;
    const uint32_t x0 = tx * TW, y0 = ty * TH;
    pdl_prologue();   // before every global load, also those of the constant per-lattice keys (tests/test_abi.py reads the SASS)
    PhiloxKey key_lat;
    if (BATCH) {
        key_lat = bv.keys[lat];
        lab16 += (size_t)lat * md.N;
        lab8 += (size_t)lat * md.N;
        in += (size_t)lat * md.N;
        out += (size_t)lat * md.N;
    }
    const PhiloxKey &key = BATCH ? key_lat : key_one;

    // one decision per open root of the tile (S3; R5 CLUSTER stream), keyed on the site index of the root
    // of its cluster in the global union-find
    const uint32_t oc = ocount[blockIdx.x];
    const uint32_t no = oc & ~WIDE_FLAG;
    const bool wide = (oc & WIDE_FLAG) != 0u;        // the tile's labels are in lab16 (two bytes per site), else in lab8
    uint32_t r = 0u;
    if (tid < no) r = groot_site_compress(parent, blockIdx.x * (uint32_t)OCAP + tid);
    uint4 lab[PASSES];                               // narrow: .x, .y hold the 8 bytes of 8 sites
    uint2 old[PASSES];
    (void)old;
#pragma unroll
    for (int c = 0; c < PASSES; ++c) {
        const uint32_t p8 = ((uint32_t)c * TILE_THREADS + tid) * 8u;
        const size_t at = (size_t)(y0 + p8 / TW) * L + x0 + p8 % TW;
        if (wide) {
            lab[c] = *reinterpret_cast<const uint4 *>(lab16 + at);
        } else {
            const uint2 b8 = *reinterpret_cast<const uint2 *>(lab8 + at);
            lab[c] = make_uint4(b8.x, b8.y, 0u, 0u);
        }
        if (MODEL == 1) old[c] = *reinterpret_cast<const uint2 *>(in + at);    // S^t (the reflection needs the old spin)
    }
    if (tid < (uint32_t)NDEC) { s_dec[DEC_BASE + tid] = (uint8_t)tid; s_dec[tid] = (uint8_t)tid; }
    for (uint32_t i = tid; i < no; i += TILE_THREADS) {
        if (i >= TILE_THREADS) r = groot_site_compress(parent, blockIdx.x * (uint32_t)OCAP + i);
        uint32_t w[4];
        philox_stream<STREAM_CLUSTER>(key, r >> 2, t, w);
        const uint32_t ww = (r & 2u) ? ((r & 1u) ? w[3] : w[2]) : ((r & 1u) ? w[1] : w[0]);
        s_dec[POS_BASE + i] = (uint8_t)(MODEL == 0 ? mulhi_q(ww, (uint32_t)md.q) : (ww >> 31));
    }
    __syncthreads();

    // S4: every site takes the decision of its root
    uint32_t m = 0u;
    if (MODEL == 1) m = axis_of_sweep(key, t, (uint32_t)md.q);
#pragma unroll
    for (int c = 0; c < PASSES; ++c) {
        const uint32_t p8 = ((uint32_t)c * TILE_THREADS + tid) * 8u;
        const size_t at = (size_t)(y0 + p8 / TW) * L + x0 + p8 % TW;
        const uint32_t w[4] = { lab[c].x, lab[c].y, lab[c].z, lab[c].w };
        uint32_t d[8];
        if (wide) {
#pragma unroll
            for (int j = 0; j < 8; ++j) d[j] = s_dec[(w[j >> 1] >> (16 * (j & 1))) & 0x3FFu];   // LOPEN | POS_BASE + pos or DEC_BASE + d
        } else {
#pragma unroll
            for (int j = 0; j < 8; ++j) d[j] = s_dec[(w[j >> 2] >> (8 * (j & 3))) & 0xFFu];     // POS_BASE + pos or d
        }
        uint2 o;
        if (MODEL == 0) {
            o.x = d[0] | (d[1] << 8) | (d[2] << 16) | (d[3] << 24);
            o.y = d[4] | (d[5] << 8) | (d[6] << 16) | (d[7] << 24);
        } else {
            const uint32_t q = (uint32_t)md.q;
            uint32_t sp[8];
#pragma unroll
            for (int j = 0; j < 8; ++j) {
                sp[j] = (((j < 4) ? old[c].x : old[c].y) >> (8 * (j & 3))) & 0xFFu;
                if (d[j]) {
                    const uint32_t vv = m + q - sp[j];          // in (0, 2q)
                    sp[j] = vv >= q ? vv - q : vv;
                }
            }
            o.x = sp[0] | (sp[1] << 8) | (sp[2] << 16) | (sp[3] << 24);
            o.y = sp[4] | (sp[5] << 8) | (sp[6] << 16) | (sp[7] << 24);
        }
        *reinterpret_cast<uint2 *>(out + at) = o;
    }
}

// Debug export (sw_get_labels): canonical root of every site.
// Sites first .. first + count - 1 -> out[0 .. count).
__global__ void k_resolve_labels(Model md, const uint16_t *lab16, const unsigned long long *parent, uint32_t first, uint32_t count,
                                 int32_t *out)
{
    const uint32_t L = (uint32_t)md.L;
    const uint32_t j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= count) return;
    const uint32_t i = first + j;
    const uint32_t y = i / L, x = i - y * L;
    const uint32_t v = lab16[i];
    // written with fuse = 0: closed -> tile-local root sp; open -> LOPEN | pos
    if (v & LOPEN) out[j] = (int32_t)groot_site(parent, ((y / TH) * (L / TW) + x / TW) * (uint32_t)OCAP + ((v & 0x3FFu) - POS_BASE));
    else out[j] = (int32_t)root_site(v, x - x % TW, y - y % TH, L);
}

// ---------------------------------------------------------------------------------------------------------
// host side
// ---------------------------------------------------------------------------------------------------------
// Tensor map of `rows` x L uint8 spins (one lattice: rows = L; a batch: its lattices stacked, rows = B * L) with a
// TW x TH box (no swizzle, no interleave).  The driver's encoder is reached through the runtime (no link against libcuda).
static inline int make_spin_map(CUtensorMap *map, const uint8_t *base, int L, size_t rows)
{
    typedef CUresult (*encode_fn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *,
                                  const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
    static encode_fn encode = nullptr;
    if (!encode) {
        void *fn = nullptr;
        cudaDriverEntryPointQueryResult qres;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres) != cudaSuccess || !fn ||
            qres != cudaDriverEntryPointSuccess)
            return -1;
        encode = reinterpret_cast<encode_fn>(fn);
    }
    const cuuint64_t dims[2] = { (cuuint64_t)L, (cuuint64_t)rows };   // innermost first
    const cuuint64_t strides[1] = { (cuuint64_t)L };                  // bytes between rows
    const cuuint32_t box[2] = { (cuuint32_t)TW, (cuuint32_t)TH };
    const cuuint32_t estr[2] = { 1u, 1u };
    const CUresult r = encode(map, CU_TENSOR_MAP_DATA_TYPE_UINT8, 2u, const_cast<uint8_t *>(base), dims, strides, box, estr,
                              CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                              CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS ? 0 : -1;
}

// Workspace of nlat lattices (labels, seam masks, edge labels, open counts), carved from ws; the union-find nodes
// (nlat * tiles * OCAP * 8 bytes) are the caller's.
static inline size_t tiled_workspace_bytes_n(int L, size_t nlat)
{
    if (!tiled_supported(L)) return 0;
    const size_t N = (size_t)L * L;
    const size_t tiles = (size_t)(L / TW) * (L / TH);
    return nlat * 2 * N + 1024 + nlat * N + 1024 + nlat * (size_t)(L / TW) * (L / 32) * 4 + 1024 + nlat * (size_t)(L / TH) * (L / 32) * 4 + 1024 +
           nlat * tiles * ECNT * 2 + 1024 + nlat * tiles * 4 + 1024;
}

static inline int tiled_init(TiledState &st, const Model &md, char *ws, const uint8_t *spins_a, const uint8_t *spins_b, size_t nlat = 1)
{
    const size_t L = (size_t)md.L;
    st.L = md.L;
    st.nlat = (uint32_t)nlat;
    st.map_base[0] = spins_a;
    st.map_base[1] = spins_b;
    if (make_spin_map(&st.map[0], spins_a, md.L, nlat * L) != 0 || make_spin_map(&st.map[1], spins_b, md.L, nlat * L) != 0) return -1;
    size_t off = 0;
    st.lab16 = reinterpret_cast<uint16_t *>(ws);
    off += (nlat * 2 * L * L + 1023) / 1024 * 1024;
    st.lab8 = reinterpret_cast<uint8_t *>(ws + off);
    off += (nlat * L * L + 1023) / 1024 * 1024;
    st.hedge = reinterpret_cast<uint32_t *>(ws + off);
    off += (nlat * (L / TW) * (L / 32) * 4 + 1023) / 1024 * 1024;
    st.vedge = reinterpret_cast<uint32_t *>(ws + off);
    off += (nlat * (L / TH) * (L / 32) * 4 + 1023) / 1024 * 1024;
    const size_t tiles = (L / TW) * (L / TH);
    st.edges = reinterpret_cast<uint16_t *>(ws + off);
    off += (nlat * tiles * ECNT * 2 + 1023) / 1024 * 1024;
    st.ocount = reinterpret_cast<uint32_t *>(ws + off);
    st.bv.tiles_per_lattice = (uint32_t)tiles;
    return 0;
}

constexpr int TILED_NUM_KERNELS = 3;
static const char *const TILED_KERNELS[TILED_NUM_KERNELS] = { "k_tile_label", "k_seam_merge", "k_tile_flip" };

// st.batch: the BATCH instantiations over st.nlat lattices (keys, thresholds and tables from st.bv; `key` and the
// thresholds inside `md` are then unused).
static inline cudaError_t tiled_launch_label(TiledState &st, const Model &md, const PhiloxKey &key, uint32_t t, const uint8_t *in,
                                      unsigned long long *parent, int fuse, cudaStream_t stream, unsigned long long *stats,
                                      unsigned long long *obs = nullptr)
{
    const uint32_t tiles = ((uint32_t)md.L / TW) * ((uint32_t)md.L / TH) * st.nlat;
    if (g_pdl_dynamic_smem) {      // occupancy experiments only
        cudaFuncSetAttribute(k_tile_label<0, false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)g_pdl_dynamic_smem);
        cudaFuncSetAttribute(k_tile_label<1, false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)g_pdl_dynamic_smem);
    }
    const int which = in == st.map_base[0] ? 0 : in == st.map_base[1] ? 1 : -1;
    if (which < 0) return cudaErrorInvalidValue;     // a spin buffer without a tensor map
    const CUtensorMap &tm = st.map[which];
    unsigned long long *const none = nullptr;
    if (st.batch) {
        if (md.model == 0)
            return launch_pdl(k_tile_label<0, false, true>, tiles, TILE_THREADS, stream, md, key, t, in, tm, st.lab16, st.lab8, parent, st.hedge,
                              st.vedge, st.edges, st.ocount, fuse, stats, none, st.bv);
        return launch_pdl(k_tile_label<1, false, true>, tiles, TILE_THREADS, stream, md, key, t, in, tm, st.lab16, st.lab8, parent, st.hedge,
                          st.vedge, st.edges, st.ocount, fuse, stats, none, st.bv);
    }
    if (stats && !st.batch) {          // counters on: the STATS instantiation (the caller does not fuse observables then)
        if (md.model == 0)
            return launch_pdl(k_tile_label<0, false, false, true>, tiles, TILE_THREADS, stream, md, key, t, in, tm, st.lab16, st.lab8, parent,
                              st.hedge, st.vedge, st.edges, st.ocount, fuse, stats, none, st.bv);
        return launch_pdl(k_tile_label<1, false, false, true>, tiles, TILE_THREADS, stream, md, key, t, in, tm, st.lab16, st.lab8, parent,
                          st.hedge, st.vedge, st.edges, st.ocount, fuse, stats, none, st.bv);
    }
    if (md.model == 0 && md.q == 2 && obs)
        return launch_pdl(k_tile_label<0, true, false>, tiles, TILE_THREADS, stream, md, key, t, in, tm, st.lab16, st.lab8, parent, st.hedge,
                          st.vedge, st.edges, st.ocount, fuse, stats, obs, st.bv);
    if (md.model == 0)
        return launch_pdl(k_tile_label<0, false, false>, tiles, TILE_THREADS, stream, md, key, t, in, tm, st.lab16, st.lab8, parent, st.hedge,
                          st.vedge, st.edges, st.ocount, fuse, stats, none, st.bv);
    return launch_pdl(k_tile_label<1, false, false>, tiles, TILE_THREADS, stream, md, key, t, in, tm, st.lab16, st.lab8, parent, st.hedge,
                      st.vedge, st.edges, st.ocount, fuse, stats, none, st.bv);
}

static inline cudaError_t tiled_launch_merge(TiledState &st, const Model &md, unsigned long long *parent, cudaStream_t stream,
                                             unsigned long long *stats)
{
    const uint32_t L = (uint32_t)md.L;
    const uint32_t ne = ((L / TW) * L + (L / TH) * L) * st.nlat;
    return launch_pdl(k_seam_merge, (ne + SEAM_THREADS - 1) / SEAM_THREADS, SEAM_THREADS, stream, md, st.hedge, st.vedge, st.edges, parent,
                      stats, st.nlat);
}

// One sweep: in = S^t (left untouched), out = S^{t+1}.  ev (optional): ev[0] is recorded before the first kernel,
// ev[k+1] after kernel k.
// obs (optional, zeroed row of the record ring): K1 adds the observables of S^t to it when it can (tiled_fuses_observables).
static inline bool tiled_fuses_observables(const Model &md) { return md.model == 0 && md.q == 2; }

static inline int tiled_sweep(TiledState &st, const Model &md, const PhiloxKey &key, uint32_t t, const uint8_t *in,
                              uint8_t *out, unsigned long long *parent, cudaStream_t stream, unsigned long long *stats,
                              uint64_t *launches, cudaEvent_t *ev, unsigned long long *obs = nullptr)
{
    const uint32_t L = (uint32_t)md.L;
    const uint32_t tiles = (L / TW) * (L / TH) * st.nlat;
    if (ev) cudaEventRecord(ev[0], stream);
    cudaError_t e = tiled_launch_label(st, md, key, t, in, parent, 1, stream, stats, obs);
    if (e != cudaSuccess) return -1;
    if (ev) cudaEventRecord(ev[1], stream);
    e = tiled_launch_merge(st, md, parent, stream, stats);
    if (e != cudaSuccess) return -1;
    if (ev) cudaEventRecord(ev[2], stream);
    if (st.batch)
        e = md.model == 0 ? launch_pdl(k_tile_flip<0, true>, tiles, TILE_THREADS, stream, md, key, t, st.lab16, st.lab8, parent, st.ocount, in, out, st.bv)
                          : launch_pdl(k_tile_flip<1, true>, tiles, TILE_THREADS, stream, md, key, t, st.lab16, st.lab8, parent, st.ocount, in, out, st.bv);
    else
        e = md.model == 0 ? launch_pdl(k_tile_flip<0, false>, tiles, TILE_THREADS, stream, md, key, t, st.lab16, st.lab8, parent, st.ocount, in, out, st.bv)
                          : launch_pdl(k_tile_flip<1, false>, tiles, TILE_THREADS, stream, md, key, t, st.lab16, st.lab8, parent, st.ocount, in, out, st.bv);
    if (e != cudaSuccess) return -1;
    if (ev) cudaEventRecord(ev[3], stream);
    *launches += 3;
    return cudaPeekAtLastError() == cudaSuccess ? 0 : -1;
}

// Debug export (sw_get_labels): label the configuration `in` with the bonds of sweep t again, this time keeping the
// tile-local root of every site (no fused decisions), merge, and resolve every site to its canonical root.
static inline int tiled_relabel(TiledState &st, const Model &md, const PhiloxKey &key, uint32_t t, const uint8_t *in,
                                unsigned long long *parent, cudaStream_t stream, uint64_t *launches)
{
    if (tiled_launch_label(st, md, key, t, in, parent, 0, stream, nullptr) != cudaSuccess) return -1;
    if (tiled_launch_merge(st, md, parent, stream, nullptr) != cudaSuccess) return -1;
    *launches += 2;
    return cudaPeekAtLastError() == cudaSuccess ? 0 : -1;
}

// ... and resolve sites first .. first + count - 1 to their canonical roots, out[0 .. count).
static inline int tiled_resolve_chunk(TiledState &st, const Model &md, const unsigned long long *parent, uint32_t first, uint32_t count,
                                      int32_t *out, cudaStream_t stream, uint64_t *launches)
{
    k_resolve_labels<<<(count + 255) / 256, 256, 0, stream>>>(md, st.lab16, parent, first, count, out);
    *launches += 1;
    return cudaPeekAtLastError() == cudaSuccess ? 0 : -1;
}

}  // namespace sw

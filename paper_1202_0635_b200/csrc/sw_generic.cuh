// Generic back-end (SW_ALGO_GENERIC): whole-lattice kernels that work for any L >= 2.
//   k_init_spins      S^0 from the INIT stream                         (R12)
//   k_bonds           S1: two bond bits per site                       (R1, R4, R5, R6)
//   k_label_init/k_union/k_flatten   S2: lock-free union-find by minimum index in global memory
//                                    (the "proper label ... smallest")
//   k_flip            S3+S4: decision from the CLUSTER stream keyed on the root, spin update
//                                                                      (R4, R9)
//   k_observables     S5: integer histograms                           (R11)
// It is the slow, simple path: the tiled back-end replaces S1/S2/S3 for L % 128 == 0 and is checked
// against this one on the device as well as against the oracle.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include "sw_philox.cuh"

namespace sw {

// Programmatic dependent launch: every kernel of the sweep lets the next one be scheduled early (its CTAs become
// resident while this grid drains) and itself waits here until the previous grid has completed and flushed.
__device__ __forceinline__ void pdl_prologue()
{
    asm volatile("griddepcontrol.launch_dependents;");
    asm volatile("griddepcontrol.wait;" ::: "memory");
}

// Occupancy experiments only (SW_DUMMY_SMEM environment variable, read once by sw_create): unused dynamic shared memory
// added to every PDL launch, to lower the number of resident CTAs per SM without touching the code.
static unsigned g_pdl_dynamic_smem = 0;

template <typename... Params, typename... Args>
static inline cudaError_t launch_pdl(void (*kernel)(Params...), unsigned grid, unsigned block, cudaStream_t stream, Args... args)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(grid);
    cfg.blockDim = dim3(block);
    cfg.dynamicSmemBytes = g_pdl_dynamic_smem;
    cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kernel, static_cast<Params>(args)...);
}

struct Model {
    int L;
    int q;
    int model;            // 0 Potts, 1 clock
    uint32_t N;           // L*L
    uint32_t thr_potts;   // floor(p 2^32), Potts
    const uint32_t *table;  // device, (2q)^2 words, clock (also valid for Potts: q*q layout unused)
};

__device__ __forceinline__ uint32_t clock_c(uint32_t s, uint32_t m, uint32_t q2)
{
    // c = (2 s - m) mod 2q, s < q, m < q  ->  2s - m + 2q in (q, 4q)
    uint32_t c = 2u * s + q2 - m;
    return c >= q2 ? c - q2 : c;
}

// the same for the four spins of a word (bytes < q <= 16): 2 s + 2q - m <= 62 per byte, no carry between bytes
__device__ __forceinline__ uint32_t clock_c4(uint32_t w, uint32_t m, uint32_t q2)
{
    const uint32_t t = 2u * w + (q2 - m) * 0x01010101u;
    const uint32_t ge = (t + (0x80u - q2) * 0x01010101u) & 0x80808080u;   // bit 7 of a byte set <=> byte >= 2q
    return t - (ge >> 7) * q2;
}

static __global__ void k_init_spins(Model md, PhiloxKey key, uint8_t *__restrict__ spins)
{
    const uint32_t g = blockIdx.x * blockDim.x + threadIdx.x;  // group of 4 sites
    const uint32_t base = g * 4u;
    if (base >= md.N) return;
    uint32_t w[4];
    philox_stream<STREAM_INIT>(key, g, 0u, w);
#pragma unroll
    for (int k = 0; k < 4; ++k)
        if (base + k < md.N) spins[base + k] = (uint8_t)mulhi_q(w[k], (uint32_t)md.q);
}

// One thread per pair of sites (2p, 2p+1): one Philox call gives the four words of the pair.
static __global__ void k_bonds(Model md, PhiloxKey key, uint32_t t, const uint8_t *__restrict__ spins,
                        uint8_t *__restrict__ bonds)
{
    const uint32_t p = blockIdx.x * blockDim.x + threadIdx.x;
    if (2u * p >= md.N) return;
    uint32_t w[4];
    philox_stream<STREAM_BOND>(key, p, t, w);
    const uint32_t q2 = 2u * (uint32_t)md.q;
    uint32_t m = 0u;
    if (md.model == 1) m = axis_of_sweep(key, t, (uint32_t)md.q);
#pragma unroll
    for (int k = 0; k < 2; ++k) {
        const uint32_t i = 2u * p + k;
        if (i >= md.N) break;
        const uint32_t y = i / (uint32_t)md.L, x = i - y * (uint32_t)md.L;
        const uint32_t xr = (x + 1u == (uint32_t)md.L) ? 0u : x + 1u;
        const uint32_t yd = (y + 1u == (uint32_t)md.L) ? 0u : y + 1u;
        const uint32_t s = spins[i];
        const uint32_t sn[2] = { spins[y * md.L + xr], spins[yd * md.L + x] };
        uint32_t b = 0u;
#pragma unroll
        for (int d = 0; d < 2; ++d) {
            uint32_t thr;
            if (md.model == 0) thr = (s == sn[d]) ? md.thr_potts : 0u;
            else thr = md.table[clock_c(s, m, q2) * q2 + clock_c(sn[d], m, q2)];
            b |= (w[2 * k + d] < thr) ? (1u << d) : 0u;
        }
        bonds[i] = (uint8_t)b;
    }
}

static __global__ void k_label_init(uint32_t N, int32_t *__restrict__ labels)
{
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < N) labels[i] = (int32_t)i;
}

// Union-find by minimum index on an int32 parent array in global memory.  Parents only ever decrease,
// so a stale read is still an ancestor and the atomicMin re-validates the root.
__device__ __forceinline__ int32_t uf_find(const int32_t *lab, int32_t a)
{
    int32_t p;
    while ((p = __ldcg(lab + a)) != a) a = p;
    return a;
}

// find with path halving: every node passed on the way is re-pointed to its grandparent.  A racing atomicMin or
// another halving store can only replace an ancestor by another ancestor, so connectivity is kept.  Loads may be
// served by a stale L1 line: a stale parent is still an ancestor, and a stale "root" is caught by the atomicMin
// of uf_union, which returns the true parent.  (L1-cached loads keep the hot roots of large clusters out of L2.)
__device__ __forceinline__ int32_t uf_find_halve(int32_t *lab, int32_t a)
{
    int32_t cur = lab[a];
    if (cur != a) {
        int32_t prev = a, next;
        while (cur > (next = lab[cur])) {
            lab[prev] = next;
            prev = cur;
            cur = next;
        }
    }
    return cur;
}

__device__ __forceinline__ void uf_union(int32_t *lab, int32_t a, int32_t b)
{
    for (;;) {
        a = uf_find_halve(lab, a);
        b = uf_find_halve(lab, b);
        if (a == b) return;
        if (a < b) { const int32_t tmp = a; a = b; b = tmp; }
        const int32_t old = atomicMin(lab + a, b);  // a > b
        if (old == a) return;                       // a was a root and now hangs under b
        a = old;                                    // a already had a parent: keep that parent connected to b
    }
}

static __global__ void k_union(Model md, const uint8_t *__restrict__ bonds, int32_t *labels)
{
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= md.N) return;
    const uint32_t b = bonds[i];
    if (!b) return;
    const uint32_t y = i / (uint32_t)md.L, x = i - y * (uint32_t)md.L;
    if (b & 1u) {
        const uint32_t xr = (x + 1u == (uint32_t)md.L) ? 0u : x + 1u;
        uf_union(labels, (int32_t)i, (int32_t)(y * md.L + xr));
    }
    if (b & 2u) {
        const uint32_t yd = (y + 1u == (uint32_t)md.L) ? 0u : y + 1u;
        uf_union(labels, (int32_t)i, (int32_t)(yd * md.L + x));
    }
}

static __global__ void k_flatten(uint32_t N, int32_t *labels)
{
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < N) labels[i] = uf_find(labels, (int32_t)i);
}

static __global__ void k_flip(Model md, PhiloxKey key, uint32_t t, const int32_t *__restrict__ labels,
                       uint8_t *__restrict__ spins)
{
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= md.N) return;
    const uint32_t r = (uint32_t)labels[i];
    uint32_t w[4];
    philox_stream<STREAM_CLUSTER>(key, r >> 2, t, w);
    const uint32_t ww = (r & 2u) ? ((r & 1u) ? w[3] : w[2]) : ((r & 1u) ? w[1] : w[0]);
    if (md.model == 0) {
        spins[i] = (uint8_t)mulhi_q(ww, (uint32_t)md.q);
    } else if (ww >> 31) {
        const uint32_t m = axis_of_sweep(key, t, (uint32_t)md.q);
        const uint32_t s = spins[i];
        const uint32_t v = m + (uint32_t)md.q - s;          // in (0, 2q)
        spins[i] = (uint8_t)(v >= (uint32_t)md.q ? v - (uint32_t)md.q : v);
    }
}

// S5 and the correlation histograms.  Both kernels count into per-thread private columns of a shared-memory table
// ([bin][thread]: conflict-free plain increments, no atomics -- with q = 2 a warp-wide shared atomic would serialise
// 16-fold on two addresses), four sites per thread and iteration with 32-bit loads, then one reduction per block and
// one global atomic per bin and block.  L % 4 != 0 (small odd lattices, generic back-end only) takes a plain path.
constexpr int HIST_THREADS = 256;

__device__ __forceinline__ uint32_t diff_mod_q(uint32_t s, uint32_t o, uint32_t q) { return s >= o ? s - o : s + q - o; }

// sum the NB bins over the block's threads and add them to out[0..NB)
template <int NB>
__device__ __forceinline__ void hist_flush(unsigned int (*h)[HIST_THREADS], unsigned long long *out)
{
    __syncthreads();
    const uint32_t lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
    for (uint32_t b = warp; b < (uint32_t)NB; b += HIST_THREADS / 32) {
        uint32_t v = 0u;
        for (uint32_t k = lane; k < (uint32_t)HIST_THREADS; k += 32u) v += h[b][k];
        v = __reduce_add_sync(0xFFFFFFFFu, v);
        if (lane == 0u && v) atomicAdd(out + b, (unsigned long long)v);
    }
}

// byte-wise (a - b) mod q of two words of four spins (all bytes < q <= 16)
__device__ __forceinline__ uint32_t diff4_mod_q(uint32_t a, uint32_t b, uint32_t q)
{
    uint32_t t = a + q * 0x01010101u - b;                                   // bytes in [1, 2q - 1]: no borrow between bytes
    const uint32_t ge = (t + (0x80u - q) * 0x01010101u) & 0x80808080u;      // bit 7 of a byte set <=> byte >= q
    return t - (ge >> 7) * q;
}
// number of bytes of v (all < 32) that differ from d
__device__ __forceinline__ uint32_t bytes_ne(uint32_t v, uint32_t d)
{
    return (uint32_t)__popc(((v ^ (d * 0x01010101u)) + 0x7F7F7F7Fu) & 0x80808080u);
}

// out[0..q) += bond_hist, out[16..16+q) += state_hist (unsigned long long, zeroed by the host).
// L % 4 == 0: four sites per thread and iteration, counted in registers with byte-parallel compares (one counter
// per value d < q; the loop over d is unrolled and cut off by the uniform test d < q), no shared-memory traffic.
// `spins` is written by the previous kernel of the PDL chain (k_tile_flip): no const __restrict__, so that its loads stay
// ordinary coherent loads ordered after griddepcontrol.wait (never ld.global.nc).
template <int QB>   // QB = 2, 4, 8 or 16 >= q: bound of the unrolled loops over the values d
__global__ void __launch_bounds__(HIST_THREADS) k_observables(Model md, const uint8_t *spins, unsigned long long *out)
{
    __shared__ unsigned int h[32][HIST_THREADS];
    const uint32_t tid = threadIdx.x;
    pdl_prologue();
    const uint32_t q = (uint32_t)md.q, L = (uint32_t)md.L;
    if (L % 16u == 0u) {
        uint32_t nb[16], ns[16], groups = 0u;        // bytes NOT equal to d, summed; turned into counts at the end
#pragma unroll
        for (int d = 0; d < QB; ++d) nb[d] = ns[d] = 0u;
        const uint32_t nq = md.N / 16u;              // 16 sites (one 128-bit load) per thread and iteration
        for (uint32_t g = blockIdx.x * blockDim.x + tid; g < nq; g += gridDim.x * blockDim.x) {
            const uint32_t i = 16u * g, y = i / L, x = i - y * L;
            const uint32_t yd = (y + 1u == L) ? 0u : y + 1u, xr = (x + 16u == L) ? 0u : x + 16u;
            const uint4 w4 = *reinterpret_cast<const uint4 *>(spins + i);
            const uint4 d4 = *reinterpret_cast<const uint4 *>(spins + (size_t)yd * L + x);
            const uint32_t nx = spins[(size_t)y * L + xr];
            const uint32_t w[4] = { w4.x, w4.y, w4.z, w4.w }, wd[4] = { d4.x, d4.y, d4.z, d4.w };
#pragma unroll
            for (int c = 0; c < 4; ++c) {
                const uint32_t wr = (w[c] >> 8) | ((c < 3 ? w[c < 3 ? c + 1 : 3] : nx) << 24);
                const uint32_t dh = diff4_mod_q(w[c], wr, q), dv = diff4_mod_q(w[c], wd[c], q);
#pragma unroll
                for (int d = 0; d < QB; ++d) {
                    if ((uint32_t)d < q) {
                        nb[d] += bytes_ne(dh, (uint32_t)d) + bytes_ne(dv, (uint32_t)d);
                        ns[d] += bytes_ne(w[c], (uint32_t)d);
                    }
                }
            }
            groups += 4u;
        }
        for (int b2 = 0; b2 < 32; ++b2) h[b2][tid] = 0u;
#pragma unroll
        for (int d = 0; d < QB; ++d) {
            h[d][tid] = ((uint32_t)d < q) ? 8u * groups - nb[d] : 0u;
            h[16 + d][tid] = ((uint32_t)d < q) ? 4u * groups - ns[d] : 0u;
        }
    } else {
        for (int b = 0; b < 32; ++b) h[b][tid] = 0u;
        for (uint32_t i = blockIdx.x * blockDim.x + tid; i < md.N; i += gridDim.x * blockDim.x) {
            const uint32_t y = i / L, x = i - y * L;
            const uint32_t xr = (x + 1u == L) ? 0u : x + 1u, yd = (y + 1u == L) ? 0u : y + 1u;
            const uint32_t s = spins[i];
            h[diff_mod_q(s, spins[y * L + xr], q)][tid] += 1u;
            h[diff_mod_q(s, spins[yd * L + x], q)][tid] += 1u;
            h[16u + s][tid] += 1u;
        }
    }
    hist_flush<32>(h, out);
}

// Correlation histogram at distance r (eq.(5), (6); R15): out[d] += number of pairs (i, i + r e_x)
// and (i, i + r e_y), periodic, with (S_i - S_{i+r}) mod q == d (unsigned long long, zeroed by the host).
template <int QB>
__global__ void __launch_bounds__(HIST_THREADS) k_correlation(Model md, const uint8_t *spins, uint32_t r, unsigned long long *out)
{
    __shared__ unsigned int h[16][HIST_THREADS];
    const uint32_t tid = threadIdx.x;
    pdl_prologue();
    const uint32_t q = (uint32_t)md.q, L = (uint32_t)md.L;
    if (L % 16u == 0u && r % 4u == 0u) {
        // 16 sites per thread and iteration (the distances the paper measures, L/4 and L/2, take this path)
        uint32_t nb[16], groups = 0u;
#pragma unroll
        for (int d = 0; d < QB; ++d) nb[d] = 0u;
        const uint32_t nq = md.N / 16u;
        for (uint32_t g = blockIdx.x * blockDim.x + tid; g < nq; g += gridDim.x * blockDim.x) {
            const uint32_t i = 16u * g, y = i / L, x = i - y * L;
            uint32_t yd = y + r; if (yd >= L) yd -= L;
            const uint4 w4 = *reinterpret_cast<const uint4 *>(spins + i);
            const uint4 d4 = *reinterpret_cast<const uint4 *>(spins + (size_t)yd * L + x);
            uint32_t wr[4];
#pragma unroll
            for (int c = 0; c < 4; ++c) {
                uint32_t xr = x + 4u * (uint32_t)c + r; if (xr >= L) xr -= L;
                wr[c] = *reinterpret_cast<const uint32_t *>(spins + (size_t)y * L + xr);
            }
            const uint32_t w[4] = { w4.x, w4.y, w4.z, w4.w }, wd[4] = { d4.x, d4.y, d4.z, d4.w };
#pragma unroll
            for (int c = 0; c < 4; ++c) {
                const uint32_t dh = diff4_mod_q(w[c], wr[c], q), dv = diff4_mod_q(w[c], wd[c], q);
#pragma unroll
                for (int d = 0; d < QB; ++d)
                    if ((uint32_t)d < q) nb[d] += bytes_ne(dh, (uint32_t)d) + bytes_ne(dv, (uint32_t)d);
            }
            groups += 4u;
        }
        for (int b2 = 0; b2 < 16; ++b2) h[b2][tid] = 0u;
#pragma unroll
        for (int d = 0; d < QB; ++d) h[d][tid] = ((uint32_t)d < q) ? 8u * groups - nb[d] : 0u;
    } else if (L % 4u == 0u) {
        uint32_t nb[16], groups = 0u;
#pragma unroll
        for (int d = 0; d < QB; ++d) nb[d] = 0u;
        const uint32_t nq = md.N / 4u;
        for (uint32_t g = blockIdx.x * blockDim.x + tid; g < nq; g += gridDim.x * blockDim.x) {
            const uint32_t i = 4u * g, y = i / L, x = i - y * L;
            uint32_t yd = y + r; if (yd >= L) yd -= L;
            const uint32_t w = *reinterpret_cast<const uint32_t *>(spins + i);
            const uint32_t wd = *reinterpret_cast<const uint32_t *>(spins + (size_t)yd * L + x);
            uint32_t wr;
            if (r % 4u == 0u) {
                uint32_t xr = x + r; if (xr >= L) xr -= L;
                wr = *reinterpret_cast<const uint32_t *>(spins + (size_t)y * L + xr);
            } else {
                wr = 0u;
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    uint32_t xr = x + (uint32_t)k + r; if (xr >= L) xr -= L;
                    wr |= (uint32_t)spins[(size_t)y * L + xr] << (8 * k);
                }
            }
            const uint32_t dh = diff4_mod_q(w, wr, q), dv = diff4_mod_q(w, wd, q);
            ++groups;
#pragma unroll
            for (int d = 0; d < QB; ++d)
                if ((uint32_t)d < q) nb[d] += bytes_ne(dh, (uint32_t)d) + bytes_ne(dv, (uint32_t)d);
        }
        for (int b2 = 0; b2 < 16; ++b2) h[b2][tid] = 0u;
#pragma unroll
        for (int d = 0; d < QB; ++d) h[d][tid] = ((uint32_t)d < q) ? 8u * groups - nb[d] : 0u;
    } else {
        for (int b = 0; b < 16; ++b) h[b][tid] = 0u;
        for (uint32_t i = blockIdx.x * blockDim.x + tid; i < md.N; i += gridDim.x * blockDim.x) {
            const uint32_t y = i / L, x = i - y * L;
            uint32_t xr = x + r; if (xr >= L) xr -= L;
            uint32_t yd = y + r; if (yd >= L) yd -= L;
            const uint32_t s = spins[i];
            h[diff_mod_q(s, spins[y * L + xr], q)][tid] += 1u;
            h[diff_mod_q(s, spins[yd * L + x], q)][tid] += 1u;
        }
    }
    hist_flush<16>(h, out);
}

// Validation of a configuration handed in by sw_set_spins: flag[0] = 1 if any value >= q.
static __global__ void k_check_spins(uint32_t N, uint32_t q, const uint8_t *__restrict__ spins, int *flag)
{
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < N && spins[i] >= q) *flag = 1;
}

}  // namespace sw

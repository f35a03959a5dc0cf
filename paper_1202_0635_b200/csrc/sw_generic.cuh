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
#include <stdint.h>
#include "sw_philox.cuh"

namespace sw {

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

__global__ void k_init_spins(Model md, PhiloxKey key, uint8_t *__restrict__ spins)
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
__global__ void k_bonds(Model md, PhiloxKey key, uint32_t t, const uint8_t *__restrict__ spins,
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

__global__ void k_label_init(uint32_t N, int32_t *__restrict__ labels)
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

__global__ void k_union(Model md, const uint8_t *__restrict__ bonds, int32_t *labels)
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

__global__ void k_flatten(uint32_t N, int32_t *labels)
{
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < N) labels[i] = uf_find(labels, (int32_t)i);
}

__global__ void k_flip(Model md, PhiloxKey key, uint32_t t, const int32_t *__restrict__ labels,
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

// S5.  out[0..q) += bond_hist, out[16..16+q) += state_hist (unsigned long long, zeroed by the host).
// Per-warp private shared-memory histograms, then one global atomic per bin per block.
__global__ void __launch_bounds__(256) k_observables(Model md, const uint8_t *__restrict__ spins,
                                                     unsigned long long *__restrict__ out)
{
    __shared__ unsigned int h[8][32];
    const int warp = threadIdx.x >> 5;
    for (int k = threadIdx.x; k < 8 * 32; k += blockDim.x) (&h[0][0])[k] = 0u;
    __syncthreads();
    const uint32_t q = (uint32_t)md.q;
    for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < md.N; i += gridDim.x * blockDim.x) {
        const uint32_t y = i / (uint32_t)md.L, x = i - y * (uint32_t)md.L;
        const uint32_t xr = (x + 1u == (uint32_t)md.L) ? 0u : x + 1u;
        const uint32_t yd = (y + 1u == (uint32_t)md.L) ? 0u : y + 1u;
        const uint32_t s = spins[i];
        const uint32_t sr = spins[y * md.L + xr], sd = spins[yd * md.L + x];
        const uint32_t d0 = s >= sr ? s - sr : s + q - sr;
        const uint32_t d1 = s >= sd ? s - sd : s + q - sd;
        atomicAdd(&h[warp][d0], 1u);
        atomicAdd(&h[warp][d1], 1u);
        atomicAdd(&h[warp][16u + s], 1u);
    }
    __syncthreads();
    if (threadIdx.x < 32) {
        unsigned long long s = 0;
        for (int w2 = 0; w2 < 8; ++w2) s += h[w2][threadIdx.x];
        if (s) atomicAdd(out + threadIdx.x, s);
    }
}

// Correlation histogram at distance r (eq.(5), (6); R15): out[d] += number of pairs (i, i + r e_x)
// and (i, i + r e_y), periodic, with (S_i - S_{i+r}) mod q == d (unsigned long long, zeroed by the host).
// Four sites per thread along x (one 32-bit load each for the site word, the word at x + r when r % 4 == 0, and the
// word r rows below); per-warp private shared-memory bins, then one global atomic per bin and block.
__global__ void __launch_bounds__(256) k_correlation(Model md, const uint8_t *__restrict__ spins, uint32_t r,
                                                     unsigned long long *__restrict__ out)
{
    __shared__ unsigned int h[8][16];
    const int warp = threadIdx.x >> 5;
    for (int k = threadIdx.x; k < 8 * 16; k += blockDim.x) (&h[0][0])[k] = 0u;
    __syncthreads();
    const uint32_t q = (uint32_t)md.q, L = (uint32_t)md.L;
    if (L % 4u == 0u) {
        const uint32_t nq = md.N / 4u;
        for (uint32_t g = blockIdx.x * blockDim.x + threadIdx.x; g < nq; g += gridDim.x * blockDim.x) {
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
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                const uint32_t s = (w >> (8 * k)) & 0xFFu, sr = (wr >> (8 * k)) & 0xFFu, sd = (wd >> (8 * k)) & 0xFFu;
                atomicAdd(&h[warp][s >= sr ? s - sr : s + q - sr], 1u);
                atomicAdd(&h[warp][s >= sd ? s - sd : s + q - sd], 1u);
            }
        }
    } else {
        for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < md.N; i += gridDim.x * blockDim.x) {
            const uint32_t y = i / L, x = i - y * L;
            uint32_t xr = x + r; if (xr >= L) xr -= L;
            uint32_t yd = y + r; if (yd >= L) yd -= L;
            const uint32_t s = spins[i], sr = spins[y * L + xr], sd = spins[yd * L + x];
            atomicAdd(&h[warp][s >= sr ? s - sr : s + q - sr], 1u);
            atomicAdd(&h[warp][s >= sd ? s - sd : s + q - sd], 1u);
        }
    }
    __syncthreads();
    if (threadIdx.x < 16) {
        unsigned long long s = 0;
        for (int w2 = 0; w2 < 8; ++w2) s += h[w2][threadIdx.x];
        if (s) atomicAdd(out + threadIdx.x, s);
    }
}

// Validation of a configuration handed in by sw_set_spins: flag[0] = 1 if any value >= q.
__global__ void k_check_spins(uint32_t N, uint32_t q, const uint8_t *__restrict__ spins, int *flag)
{
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < N && spins[i] >= q) *flag = 1;
}

}  // namespace sw

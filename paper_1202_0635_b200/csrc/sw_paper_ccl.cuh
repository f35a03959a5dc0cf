// The paper's own two cluster labellers as selectable A/B back-ends (NEXT-4 of the scope table), written from the
// text of PAPER.md:53-67 (Figs 1 and 2 are missing from the extraction; only their captions survive):
//
//   SW_ALGO_HAWICK    "Label Equivalence" of Hawick et al.: two arrays (label, R), three kernels
//                     per iteration -- scan (every site compares its label with the labels of its bonded neighbours and
//                     lowers R[label] with atomicMin), analysis (threads with label[i] == i track R back until it stops
//                     changing), labeling (label[i] <- R[label[i]]) -- iterated until a scan changes nothing.
//   SW_ALGO_KALENTEV  the refinement of Kalentev et al.: one array, two kernels -- scan (writes the
//                     smaller neighbour label into label[label[i]], no atomics: a lost race is repaired by the next
//                     iteration) and analysis (run where label[label] != label) -- iterated until a scan changes nothing.
//
// Both converge to "every site carries the smallest site index of its cluster" (the proper label of PAPER.md:47), so the
// spins they lead to equal the oracle's bit for bit.  They are prior art kept for comparison: they re-scan the whole
// lattice 6-9 times per sweep with a host round trip per iteration, which is exactly what the tiled
// back-end avoids.  The iteration counts are reported through sw_stats next to the paper's 6.6-8.6 at Tc.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "sw_generic.cuh"

namespace sw {

// smallest label among the bonded neighbours of site i (and its own), bonds[i]: bit0 = bond to +x, bit1 = bond to +y
__device__ __forceinline__ int32_t ccl_min_neighbour(const Model &md, const uint8_t *bonds, const int32_t *label, uint32_t i, int32_t own)
{
    const uint32_t L = (uint32_t)md.L;
    const uint32_t y = i / L, x = i - y * L;
    const uint32_t xr = (x + 1u == L) ? 0u : x + 1u, xl = (x == 0u) ? L - 1u : x - 1u;
    const uint32_t yd = (y + 1u == L) ? 0u : y + 1u, yu = (y == 0u) ? L - 1u : y - 1u;
    const uint32_t b = bonds[i];
    int32_t m = own;
    if (b & 1u) m = min(m, label[y * L + xr]);
    if (b & 2u) m = min(m, label[yd * L + x]);
    if (bonds[y * L + xl] & 1u) m = min(m, label[y * L + xl]);
    if (bonds[yu * L + x] & 2u) m = min(m, label[yu * L + x]);
    return m;
}

__global__ void k_ccl_init(uint32_t N, int32_t *label, int32_t *R)
{
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    label[i] = (int32_t)i;
    if (R) R[i] = (int32_t)i;
}

// ---- Hawick et al., PAPER.md:53 -----------------------------------------------------------------------------------
__global__ void k_hawick_scan(Model md, const uint8_t *bonds, const int32_t *label, int32_t *R, int *changed)
{
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= md.N) return;
    const int32_t own = label[i];
    const int32_t m = ccl_min_neighbour(md, bonds, label, i, own);
    if (m < own) {
        atomicMin(&R[own], m);
        *changed = 1;
    }
}

__global__ void k_hawick_analysis(uint32_t N, const int32_t *label, int32_t *R)
{
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N || label[i] != (int32_t)i) return;
    int32_t r = R[i], next;
    while ((next = R[r]) != r) r = next;      // "tracks back the temporal variable until it remains unchanged"
    R[i] = r;
}

__global__ void k_hawick_labeling(uint32_t N, int32_t *label, const int32_t *R)
{
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < N) label[i] = R[label[i]];
}

// ---- Kalentev et al., PAPER.md:65-67 ------------------------------------------------------------------------------
__global__ void k_kalentev_scan(Model md, const uint8_t *bonds, int32_t *label, int *changed)
{
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= md.N) return;
    const int32_t own = label[i];
    const int32_t m = ccl_min_neighbour(md, bonds, label, i, own);
    if (m < own) {
        label[own] = m;            // no atomic: a lost race is repaired by the next iteration
        *changed = 1;
    }
}

__global__ void k_kalentev_analysis(uint32_t N, int32_t *label)
{
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    int32_t l = label[i];
    int32_t ref = label[l];
    if (ref == l) return;          // executed "when label[label] is not equal to label"
    while (ref != l) { l = ref; ref = label[l]; }
    label[i] = l;
}

// Labels of the bond configuration `bonds` into `label` by the chosen method; returns the number of iterations (scan
// passes, the terminating one included) or -1 on a CUDA error.  One host round trip per iteration, as in the paper.
static inline int paper_ccl_label(int algo_kalentev, const Model &md, const uint8_t *bonds, int32_t *label, int32_t *R, int *d_changed,
                                  cudaStream_t stream, uint64_t *launches)
{
    const unsigned bs = 256, grid = (md.N + bs - 1) / bs;
    k_ccl_init<<<grid, bs, 0, stream>>>(md.N, label, algo_kalentev ? nullptr : R);
    *launches += 1;
    for (int iter = 1;; ++iter) {
        if (cudaMemsetAsync(d_changed, 0, sizeof(int), stream) != cudaSuccess) return -1;
        if (algo_kalentev) k_kalentev_scan<<<grid, bs, 0, stream>>>(md, bonds, label, d_changed);
        else k_hawick_scan<<<grid, bs, 0, stream>>>(md, bonds, label, R, d_changed);
        *launches += 1;
        int changed = 0;
        if (cudaMemcpyAsync(&changed, d_changed, sizeof(int), cudaMemcpyDeviceToHost, stream) != cudaSuccess) return -1;
        if (cudaStreamSynchronize(stream) != cudaSuccess) return -1;
        if (!changed) return iter;
        if (algo_kalentev) {
            k_kalentev_analysis<<<grid, bs, 0, stream>>>(md.N, label);
            *launches += 1;
        } else {
            k_hawick_analysis<<<grid, bs, 0, stream>>>(md.N, label, R);
            k_hawick_labeling<<<grid, bs, 0, stream>>>(md.N, label, R);
            *launches += 2;
        }
        if (iter > 100000) return -1;
    }
}

}  // namespace sw

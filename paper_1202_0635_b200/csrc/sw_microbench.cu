// Instruction-issue probes (sw_microbench of include/sw.h).  Measurement infrastructure only: the sweep never calls
// anything in this file.  Every probe runs one CTA per SM whose warps execute a loop of ILP independent dependency
// chains of one SASS instruction (or a fixed mix) and reports how many of those warp-instructions one SM sub-partition
// (SMSP, the unit that owns a warp scheduler and one dispatch port) retires per SM clock cycle, from clock64() inside
// the kernel.  The "alu" roofline of DESIGN.md section 6 is derived from these numbers, not from a model.
#include <cuda_runtime.h>
#include <stdint.h>

#include "sw.h"
#include "sw_philox.cuh"

namespace swmb {

enum Probe : int {
    P_LOP3 = 0, P_IADD, P_SHF, P_SETP_SEL, P_CARRY_PAIR, P_FLO, P_BREV, P_POPC, P_IMAD, P_IMAD_IMM, P_IMAD_WIDE, P_IMAD_HI,
    P_MIX_LOP3_IMAD, P_MIX_LOP3_WIDE, P_MIX_2LOP3_WIDE, P_PHILOX, P_LDS, P_STS, P_SHFL, P_PRMT, P_MIX_LOP3_LDS, P_MIX_IMAD_LDS,
    P_MIX_LOP3_IMAD_LDS, P_VOTE, P_ATOMS_MIN,
    P_WIDE_IMAD, P_MIX_LOP3_HI, P_MIX_LOP3_FLO, P_MIX_IMAD_FLO, P_MIX_LOP3_SHFL, P_MIX_LDS_STS, P_I2F, P_PHILOX_HILO,
    P_PHILOX_PLUS_LOP3, P_PHILOX_HILO_PLUS_LOP3, P_ATOMS_MIN_RET, P_ATOMS_MIN_RET_1LANE, P_COUNT
};

static const char *const NAMES[P_COUNT] = {
    "LOP3", "IADD3", "SHF", "ISETP+SEL (pair)", "IADD3.CC+IADD3.X (pair)", "FLO", "BREV", "POPC", "IMAD (3 reg)", "IMAD (imm)",
    "IMAD.WIDE.U32 (imm) + LOP3 (pair, Philox half-round)", "IMAD.HI.U32", "LOP3+IMAD 1:1", "LOP3 + (IMAD.WIDE+LOP3) = 2:1", "LOP3 + (IMAD.WIDE+LOP3) = 3:1",
    "Philox4x32-10 call (one call = 1 unit)", "LDS.32", "STS.32", "SHFL.BFLY", "PRMT", "LOP3+LDS 1:1", "IMAD+LDS 1:1",
    "LOP3+IMAD+LDS 1:1:1", "VOTE.ANY (ballot)", "ATOMS.MIN (distinct addresses)",
    "IMAD.WIDE.U32 (imm) + IMAD (pair)", "LOP3+IMAD.HI 1:1", "LOP3+FLO 1:1", "IMAD+FLO 1:1", "LOP3+SHFL 1:1", "LDS+STS 1:1", "I2F.U32",
    "Philox4x32-10 call, products as IMAD.HI + IMAD (one call = 1 unit)", "Philox call + 40 independent LOP3 (one unit)",
    "Philox call (IMAD.HI + IMAD) + 40 independent LOP3 (one unit)",
    "ATOMS.MIN with return value (distinct addresses, result feeds the next)", "ATOMS.MIN with return value, one active lane per warp"
};

constexpr int ILP = 8;      // independent chains per thread
constexpr int REPS = 16;    // chain steps per loop iteration: ILP * REPS units per iteration

template <int P>
__device__ __forceinline__ void step(uint32_t &x, uint64_t &p, uint32_t a, uint32_t b, uint32_t saddr)
{
    if (P == P_LOP3) asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(x) : "r"(a), "r"(b));
    else if (P == P_IADD) asm volatile("add.u32 %0, %0, %1;" : "+r"(x) : "r"(a));
    else if (P == P_SHF) asm volatile("shf.l.wrap.b32 %0, %0, %1, 5;" : "+r"(x) : "r"(a));
    else if (P == P_SETP_SEL) asm volatile("{.reg .pred q; setp.lt.u32 q, %0, %1; selp.u32 %0, %2, %0, q;}" : "+r"(x) : "r"(a), "r"(b));
    else if (P == P_CARRY_PAIR) asm volatile("{.reg .u32 t; add.cc.u32 t, %0, %1; addc.u32 %0, %0, %0;}" : "+r"(x) : "r"(a));
    else if (P == P_FLO) asm volatile("bfind.u32 %0, %0;" : "+r"(x));
    else if (P == P_BREV) asm volatile("brev.b32 %0, %0;" : "+r"(x));
    else if (P == P_POPC) asm volatile("popc.b32 %0, %0;" : "+r"(x));
    else if (P == P_IMAD) asm volatile("mad.lo.u32 %0, %0, %1, %2;" : "+r"(x) : "r"(a), "r"(b));
    else if (P == P_IMAD_IMM) asm volatile("mad.lo.u32 %0, %0, 0x9E3779B1, %1;" : "+r"(x) : "r"(b));
    else if (P == P_IMAD_WIDE)   // one Philox half-round: 64-bit product by a constant, both halves folded back by one 3-input XOR
        asm volatile("{.reg .u32 lo, hi; .reg .u64 w; mul.wide.u32 w, %0, 0xD2511F53; mov.b64 {lo, hi}, w; lop3.b32 %0, lo, hi, %1, 0x96;}" : "+r"(x) : "r"(a));
    else if (P == P_IMAD_HI) asm volatile("mul.hi.u32 %0, %0, %1;" : "+r"(x) : "r"(a));
    else if (P == P_SHFL) asm volatile("shfl.sync.bfly.b32 %0, %0, 1, 0x1f, 0xffffffff;" : "+r"(x));
    else if (P == P_PRMT) asm volatile("prmt.b32 %0, %0, %1, 0x2103;" : "+r"(x) : "r"(a));
    else if (P == P_LDS) asm volatile("ld.volatile.shared.u32 %0, [%1];" : "=r"(x) : "r"(saddr));
    else if (P == P_STS) asm volatile("st.shared.u32 [%1], %0;" : : "r"(x), "r"(saddr));
    else if (P == P_VOTE) asm volatile("{.reg .pred q; setp.ne.u32 q, %0, 0; vote.sync.ballot.b32 %0, q, 0xffffffff;}" : "+r"(x));
    else if (P == P_WIDE_IMAD)   // x = hi(x C); the low half feeds an IMAD accumulator kept in the upper half of p
        asm volatile("{.reg .u32 lo, hi, y, z; .reg .u64 w; mov.b64 {z, y}, %1; mul.wide.u32 w, %0, 0xD2511F53; mov.b64 {lo, %0}, w; mad.lo.u32 y, lo, %2, y; mov.b64 %1, {z, y};}" : "+r"(x), "+l"(p) : "r"(a));
    else if (P == P_I2F) asm volatile("{.reg .f32 f; cvt.rn.f32.u32 f, %0; mov.b32 %0, f;}" : "+r"(x));
    else if (P == P_ATOMS_MIN_RET) asm volatile("atom.shared.min.u32 %0, [%1], %0;" : "+r"(x) : "r"(saddr));
    else if (P == P_ATOMS_MIN_RET_1LANE) { if ((threadIdx.x & 31u) == 0u) asm volatile("atom.shared.min.u32 %0, [%1], %0;" : "+r"(x) : "r"(saddr)); }
    else if (P == P_ATOMS_MIN) asm volatile("{.reg .u32 t; atom.shared.min.u32 t, [%1], %0;}" : : "r"(x), "r"(saddr));
}

// units of the probe per chain step (pairs count once; the mixes alternate over the chains instead)
template <int P>
__global__ void __launch_bounds__(1024) k_probe(int iters, uint32_t a, uint32_t b, sw::PhiloxKey key, unsigned long long *cycles,
                                                uint32_t *sink)
{
    __shared__ uint32_t s_buf[1024 * 2];
    __shared__ unsigned long long s_t0, s_t1;
    const uint32_t tid = threadIdx.x;
    s_buf[tid] = tid; s_buf[tid + 1024] = a;
    if (tid == 0) { s_t0 = ~0ull; s_t1 = 0ull; }
    __syncthreads();
    uint32_t x[ILP];
    uint64_t p[ILP];
#pragma unroll
    for (int j = 0; j < ILP; ++j) { x[j] = a * (tid + 1u) + (uint32_t)j * b; p[j] = ((uint64_t)x[j] << 32) | (tid + 7u); }
    const uint32_t saddr = (uint32_t)__cvta_generic_to_shared(s_buf + tid);   // one bank per lane: conflict-free
    const unsigned long long t0 = clock64();
#pragma unroll 1
    for (int it = 0; it < iters; ++it) {
        if (P == P_PHILOX || P == P_PHILOX_HILO || P == P_PHILOX_PLUS_LOP3 || P == P_PHILOX_HILO_PLUS_LOP3) {
            constexpr bool HILO = (P == P_PHILOX_HILO || P == P_PHILOX_HILO_PLUS_LOP3);
            constexpr bool PLUS = (P == P_PHILOX_PLUS_LOP3 || P == P_PHILOX_HILO_PLUS_LOP3);
#pragma unroll
            for (int j = 0; j < ILP / 2; ++j) {       // chains 0..3: Philox; chains 4..7: the independent LOP3 filler
                uint32_t w[4];
                if (!HILO) {
                    sw::philox_stream<sw::STREAM_BOND, 0u>(key, x[j], (uint32_t)it, w);
                } else {
                    uint32_t x0 = x[j], x1 = (uint32_t)it, x2 = 0u, x3 = 0u;
#pragma unroll
                    for (int r = 0; r < 10; ++r) {
                        uint32_t h0, l0, h1, l1;
                        asm volatile("mul.hi.u32 %0, %1, %2;" : "=r"(h0) : "r"(x0), "r"(a));      // a, b = the two multipliers, in registers, so
                        asm volatile("mul.lo.u32 %0, %1, 0xD2511F53;" : "=r"(l0) : "r"(x0));
                        asm volatile("mul.hi.u32 %0, %1, %2;" : "=r"(h1) : "r"(x2), "r"(b));      // that ptxas cannot fuse hi and lo into IMAD.WIDE
                        asm volatile("mul.lo.u32 %0, %1, 0xCD9E8D57;" : "=r"(l1) : "r"(x2));
                        const uint32_t y0 = h1 ^ x1 ^ key.rk0[r], y2 = h0 ^ x3 ^ key.rk1[r];
                        x1 = l1; x3 = l0; x0 = y0; x2 = y2;
                    }
                    w[0] = x0; w[1] = x1; w[2] = x2; w[3] = x3;
                }
                x[j] = w[0] ^ w[1] ^ w[2] ^ w[3];     // 2 more LOP3 per call
                if (PLUS) {
#pragma unroll
                    for (int r = 0; r < 10; ++r) step<P_LOP3>(x[4 + j], p[j], a, b, saddr);
                }
            }
        } else {
#pragma unroll
            for (int r = 0; r < REPS; ++r) {
#pragma unroll
                for (int j = 0; j < ILP; ++j) {
                    if (P == P_MIX_LOP3_IMAD) { if (j & 1) step<P_IMAD>(x[j], p[j], a, b, saddr); else step<P_LOP3>(x[j], p[j], a, b, saddr); }
                    else if (P == P_MIX_LOP3_WIDE) { if (j & 1) step<P_IMAD_WIDE>(x[j], p[j], a, b, saddr); else step<P_LOP3>(x[j], p[j], a, b, saddr); }
                    else if (P == P_MIX_2LOP3_WIDE) {
                        // chains 0..5 of 8: LOP3 on 0,1,3,4,6,7 ... keep exactly 2:1 over chains 0..5, chains 6,7 idle
                        if (j < 6) { if (j % 3 == 2) step<P_IMAD_WIDE>(x[j], p[j], a, b, saddr); else step<P_LOP3>(x[j], p[j], a, b, saddr); }
                    }
                    else if (P == P_MIX_LOP3_HI) { if (j & 1) step<P_IMAD_HI>(x[j], p[j], a, b, saddr); else step<P_LOP3>(x[j], p[j], a, b, saddr); }
                    else if (P == P_MIX_LOP3_FLO) { if (j & 1) step<P_FLO>(x[j], p[j], a, b, saddr); else step<P_LOP3>(x[j], p[j], a, b, saddr); }
                    else if (P == P_MIX_IMAD_FLO) { if (j & 1) step<P_FLO>(x[j], p[j], a, b, saddr); else step<P_IMAD>(x[j], p[j], a, b, saddr); }
                    else if (P == P_MIX_LOP3_SHFL) { if (j & 1) step<P_SHFL>(x[j], p[j], a, b, saddr); else step<P_LOP3>(x[j], p[j], a, b, saddr); }
                    else if (P == P_MIX_LDS_STS) { if (j & 1) step<P_STS>(x[j], p[j], a, b, saddr + 4096u); else step<P_LDS>(x[j], p[j], a, b, saddr); }
                    else if (P == P_MIX_LOP3_LDS) { if (j & 1) step<P_LDS>(x[j], p[j], a, b, saddr + 4096u * (uint32_t)(j >> 2)); else step<P_LOP3>(x[j], p[j], a, b, saddr); }
                    else if (P == P_MIX_IMAD_LDS) { if (j & 1) step<P_LDS>(x[j], p[j], a, b, saddr + 4096u * (uint32_t)(j >> 2)); else step<P_IMAD>(x[j], p[j], a, b, saddr); }
                    else if (P == P_MIX_LOP3_IMAD_LDS) {
                        if (j < 6) {
                            if (j % 3 == 0) step<P_LOP3>(x[j], p[j], a, b, saddr);
                            else if (j % 3 == 1) step<P_IMAD>(x[j], p[j], a, b, saddr);
                            else step<P_LDS>(x[j], p[j], a, b, saddr + 4096u * (uint32_t)(j >> 2));
                        }
                    }
                    else if (P == P_IADD) asm volatile("add.u32 %0, %0, %1;" : "+r"(x[j]) : "r"(x[(j + 1) % ILP]));   // cannot be folded
                    else step<P>(x[j], p[j], a, b, saddr + ((P == P_LDS || P == P_STS) ? 4096u * (uint32_t)(j & 1) : 0u));
                }
            }
        }
    }
    const unsigned long long t1 = clock64();
    atomicMin(&s_t0, t0);
    atomicMax(&s_t1, t1);
    uint32_t acc = 0u;
#pragma unroll
    for (int j = 0; j < ILP; ++j) acc ^= x[j] ^ (uint32_t)p[j] ^ (uint32_t)(p[j] >> 32);
    if (acc == 0x12345u) sink[0] = acc;      // keeps every chain alive
    __syncthreads();
    if (tid == 0) cycles[blockIdx.x] = s_t1 - s_t0;
}

template <int P>
static cudaError_t run(int grid, int block, int iters, const sw::PhiloxKey &key, unsigned long long *d_cyc, uint32_t *d_sink)
{
    const bool hilo = (P == P_PHILOX_HILO || P == P_PHILOX_HILO_PLUS_LOP3);
    k_probe<P><<<grid, block>>>(iters, hilo ? 0xD2511F53u : 0x9E3779B9u, hilo ? 0xCD9E8D57u : 0x7F4A7C15u, key, d_cyc, d_sink);
    return cudaGetLastError();
}

static double units_per_iter(int probe)
{
    switch (probe) {
    case P_PHILOX: case P_PHILOX_HILO: return ILP / 2;
    case P_PHILOX_PLUS_LOP3: case P_PHILOX_HILO_PLUS_LOP3: return ILP / 2;
    case P_MIX_2LOP3_WIDE: return 8.0 * REPS;   // 6 chains: 4 LOP3 + 2 pairs = 8 warp-instructions per step
    case P_MIX_LOP3_WIDE: return 12.0 * REPS;   // 8 chains: 4 LOP3 + 4 pairs = 12 warp-instructions per step
    case P_MIX_LOP3_IMAD_LDS: return 6.0 * REPS;
    default: return (double)ILP * REPS;
    }
}

}  // namespace swmb

extern "C" {

const char *sw_microbench_name(int probe)
{
    return (probe >= 0 && probe < swmb::P_COUNT) ? swmb::NAMES[probe] : nullptr;
}

int sw_microbench(int probe, int warps_per_smsp, int iters, double *out)
{
    using namespace swmb;
    if (probe < 0 || probe >= P_COUNT || !out || iters < 1 || warps_per_smsp < 1 || warps_per_smsp > 16) return SW_ERR_ARG;
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) {
        cudaGetLastError();
        return SW_ERR_CUDA;
    }
    // one CTA per SM with 4 * w warps (w <= 8), two CTAs per SM of 32 warps each for w = 16
    const int ctas_per_sm = warps_per_smsp > 8 ? 2 : 1;
    const int block = 128 * warps_per_smsp / ctas_per_sm;
    const int grid = sms * ctas_per_sm;
    unsigned long long *d_cyc = nullptr;
    uint32_t *d_sink = nullptr;
    if (cudaMalloc((void **)&d_cyc, 8 * (size_t)grid) != cudaSuccess || cudaMalloc((void **)&d_sink, 64) != cudaSuccess) {
        cudaFree(d_cyc);
        cudaGetLastError();
        return SW_ERR_NOMEM;
    }
    const sw::PhiloxKey key = sw::make_philox_key(0x5EEDull);
    cudaError_t e = cudaSuccess;
    for (int rep = 0; rep < 2 && e == cudaSuccess; ++rep) {      // the first run warms the instruction cache
        switch (probe) {
#define SW_MB_CASE(P) case P: e = run<P>(grid, block, iters, key, d_cyc, d_sink); break;
        SW_MB_CASE(P_LOP3) SW_MB_CASE(P_IADD) SW_MB_CASE(P_SHF) SW_MB_CASE(P_SETP_SEL) SW_MB_CASE(P_CARRY_PAIR) SW_MB_CASE(P_FLO)
        SW_MB_CASE(P_BREV) SW_MB_CASE(P_POPC) SW_MB_CASE(P_IMAD) SW_MB_CASE(P_IMAD_IMM) SW_MB_CASE(P_IMAD_WIDE) SW_MB_CASE(P_IMAD_HI)
        SW_MB_CASE(P_MIX_LOP3_IMAD) SW_MB_CASE(P_MIX_LOP3_WIDE) SW_MB_CASE(P_MIX_2LOP3_WIDE) SW_MB_CASE(P_PHILOX) SW_MB_CASE(P_LDS)
        SW_MB_CASE(P_STS) SW_MB_CASE(P_SHFL) SW_MB_CASE(P_PRMT) SW_MB_CASE(P_MIX_LOP3_LDS) SW_MB_CASE(P_MIX_IMAD_LDS)
        SW_MB_CASE(P_MIX_LOP3_IMAD_LDS) SW_MB_CASE(P_VOTE) SW_MB_CASE(P_ATOMS_MIN)
        SW_MB_CASE(P_WIDE_IMAD) SW_MB_CASE(P_MIX_LOP3_HI) SW_MB_CASE(P_MIX_LOP3_FLO) SW_MB_CASE(P_MIX_IMAD_FLO) SW_MB_CASE(P_MIX_LOP3_SHFL)
        SW_MB_CASE(P_MIX_LDS_STS) SW_MB_CASE(P_I2F) SW_MB_CASE(P_PHILOX_HILO) SW_MB_CASE(P_PHILOX_PLUS_LOP3) SW_MB_CASE(P_PHILOX_HILO_PLUS_LOP3)
        SW_MB_CASE(P_ATOMS_MIN_RET) SW_MB_CASE(P_ATOMS_MIN_RET_1LANE)
#undef SW_MB_CASE
        default: break;
        }
        if (e == cudaSuccess) e = cudaDeviceSynchronize();
    }
    int rc = SW_OK;
    if (e != cudaSuccess) {
        rc = SW_ERR_CUDA;
    } else {
        unsigned long long *h = new unsigned long long[grid];
        cudaMemcpy(h, d_cyc, 8 * (size_t)grid, cudaMemcpyDeviceToHost);
        unsigned long long mx = 0, mn = ~0ull;
        for (int k = 0; k < grid; ++k) { mx = h[k] > mx ? h[k] : mx; mn = h[k] < mn ? h[k] : mn; }
        delete[] h;
        const double units = units_per_iter(probe) * (double)iters * (double)(warps_per_smsp / ctas_per_sm);   // per SMSP and CTA
        out[0] = units * ctas_per_sm / (double)mx;   // units per cycle per SMSP (slowest CTA; w = 16: both CTAs of an SM overlap)
        out[1] = (double)mx;
        out[2] = (double)mn;
        out[3] = units * ctas_per_sm;
    }
    cudaFree(d_cyc);
    cudaFree(d_sink);
    return rc;
}

}  // extern "C"

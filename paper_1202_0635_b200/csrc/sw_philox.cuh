// Device-side Philox4x32-10 and the random streams of DESIGN.md R5 (CUDA path only; the oracle has
// its own, separate implementation in oracle/sw_oracle.c).
//
// One call turns a 128-bit counter and a 64-bit key into four 32-bit words.  The ten round keys
// (key + r * Weyl constant) depend only on the seed, so the host computes them once per context and
// hands them to every kernel by value: they live in the constant bank and feed the XOR directly.
#pragma once
#include <stdint.h>

namespace sw {

struct PhiloxKey {
    uint32_t rk0[10];  // (seed lo) + r * 0x9E3779B9
    uint32_t rk1[10];  // (seed hi) + r * 0xBB67AE85
    uint32_t m0, m1;   // the two Philox multipliers once more, as run-time values (see philox_stream)
};

static inline PhiloxKey make_philox_key(uint64_t seed)
{
    PhiloxKey k;
    uint32_t a = (uint32_t)(seed & 0xFFFFFFFFull), b = (uint32_t)(seed >> 32);
    for (int r = 0; r < 10; ++r) {
        k.rk0[r] = a;
        k.rk1[r] = b;
        a += 0x9E3779B9u;
        b += 0xBB67AE85u;
    }
    k.m0 = 0xD2511F53u;
    k.m1 = 0xCD9E8D57u;
    return k;
}

enum : uint32_t { STREAM_BOND = 0u, STREAM_CLUSTER = 1u, STREAM_AXIS = 2u, STREAM_INIT = 3u };

// Counter (c0, t, STREAM, 0).  w[0..3] receive the four output words.
//
// HILO rounds (bit r of the mask) compute the 64-bit product as IMAD.HI (multiplier read from the key, a run-time value
// ptxas cannot fuse with the immediate of the low half) + IMAD instead of one IMAD.WIDE.  Measured on B200
// (profiles/r2_microbench.md): IMAD.WIDE holds the FMA pipe for 4 cycles AND the ALU pipe for 2; IMAD.HI + IMAD hold
// the FMA pipe for 4 + 2 and leave the ALU pipe alone.  Kernels whose other work is ALU-pipe bound (the labeling
// kernel) run such rounds on the otherwise idle FMA pipe.
#ifndef SW_PHILOX_HILO_MASK
#define SW_PHILOX_HILO_MASK 0u
#endif
template <uint32_t STREAM, uint32_t HILO = SW_PHILOX_HILO_MASK>
__device__ __forceinline__ void philox_stream(const PhiloxKey &key, uint32_t c0, uint32_t t, uint32_t (&w)[4])
{
    uint32_t x0 = c0, x1 = t, x2 = STREAM, x3 = 0u;
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        uint32_t h0, l0, h1, l1;
        if ((HILO >> r) & 1u) {
            h0 = __umulhi(x0, key.m0); l0 = x0 * 0xD2511F53u;
            h1 = __umulhi(x2, key.m1); l1 = x2 * 0xCD9E8D57u;
        } else {
            const uint64_t p0 = (uint64_t)0xD2511F53u * (uint64_t)x0;
            const uint64_t p1 = (uint64_t)0xCD9E8D57u * (uint64_t)x2;
            h0 = (uint32_t)(p0 >> 32); l0 = (uint32_t)p0;
            h1 = (uint32_t)(p1 >> 32); l1 = (uint32_t)p1;
        }
        const uint32_t y0 = h1 ^ x1 ^ key.rk0[r];
        const uint32_t y2 = h0 ^ x3 ^ key.rk1[r];
        x1 = l1;
        x3 = l0;
        x0 = y0;
        x2 = y2;
    }
    w[0] = x0; w[1] = x1; w[2] = x2; w[3] = x3;
}

__device__ __forceinline__ uint32_t mulhi_q(uint32_t w, uint32_t q) { return __umulhi(w, q); }

// Mirror axis of sweep t (clock model, R4): one call, identical in every thread.
__device__ __forceinline__ uint32_t axis_of_sweep(const PhiloxKey &key, uint32_t t, uint32_t q)
{
    uint32_t w[4];
    philox_stream<STREAM_AXIS>(key, 0u, t, w);
    return mulhi_q(w[0], q);
}

}  // namespace sw

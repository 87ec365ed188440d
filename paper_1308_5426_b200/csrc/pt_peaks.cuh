// pt_peaks.cuh -- instruction-rate micro-benchmarks behind pt_measure_peaks (include/pt.h).
//
// The roofline of the direct sweep kernel is an ALU roofline: its denominator is the rate at
// which one SM issues IDP.2A (two 16-bit x 8-bit multiply-accumulates per lane).  SURVEY.md H7 makes measuring that
// rate the builder's duty: these kernels measure it, alone and in the instruction mix of the bulk loop (one PRMT table
// look-up per two IDP.2A), next to IDP.4A, IMAD, PRMT, LOP3 and the shared-memory load rate, for 1..4 warps per SM
// sub-partition.  Rates are per SM and per clock, taken with clock64() inside the kernel (independent of the SM clock).
#pragma once
#include <cstdint>

namespace ptk {

enum PeakPattern {
    PEAK_IDP2A = 0,        // IDP.2A only
    PEAK_IDP4A = 1,        // IDP.4A only
    PEAK_IMAD = 2,         // IMAD only
    PEAK_PRMT = 3,         // PRMT only
    PEAK_LOP3 = 4,         // LOP3 only
    PEAK_MIX_BULK = 5,     // 1 PRMT + 2 IDP.2A (the bulk loop's mix); rate counts IDP.2A only
    PEAK_MIX_LOP = 6,      // 1 LOP3 + 2 IDP.2A; rate counts IDP.2A only
    PEAK_LDS128 = 7,       // LDS.128 (conflict-free); rate in bytes per clock
    PEAK_MIX_BULK4 = 8,    // 1 PRMT + 4 IDP.2A (both coupling halves); rate counts IDP.2A only
    PEAK_MIX_MIRROR = 9,   // 2 PRMT + 1 ADD + 2 IDP.2A (mirror-paired pair terms, 8 per group); rate counts IDP.2A only
    PEAK_TILE_NEAR = 10,   // the bulk tile of sweep_direct_kernel as it stands: 8 sites x 16 steps, per step and site one
                           // PRMT on the site's two table registers and two IDP.2A on packed coupling registers (39 of
                           // them, as in the kernel); rate counts IDP.2A only
    PEAK_TILE_FAR = 11,    // the same tile in the far form (PT_FAR): one PRMT and ONE IDP.4A per step and site; rate counts
                           // the IDP.4A (each covers the four pair terms that take two IDP.2A in the near form)
    PEAK_N = 12
};

constexpr int PEAK_UNROLL = 16;   // independent dependency chains per thread
constexpr int PEAK_ITERS = 512;
constexpr int PEAK_TILE_ITERS = 64;   // tiles (8 sites x 16 steps = 128 look-ups) per thread in the tile patterns

// out[blockIdx.x] = clocks the CTA needed; sink keeps the results alive.
template <int PATTERN>
__global__ void __launch_bounds__(512, 1) peak_kernel(long long* __restrict__ clocks, uint32_t* __restrict__ sink,
                                                      uint32_t seed) {
    __shared__ __align__(16) uint32_t s_buf[512 * 4];
    const int tid = threadIdx.x;
    for (int n = tid; n < 512 * 4; n += blockDim.x) s_buf[n] = seed + n;
    uint32_t acc[PEAK_UNROLL], a[PEAK_UNROLL], b[PEAK_UNROLL];
#pragma unroll
    for (int i = 0; i < PEAK_UNROLL; ++i) {
        acc[i] = seed * (i + 1) + tid;
        a[i] = (seed ^ (0x9E3779B9u * (i + 1))) + tid;
        b[i] = (seed + 0x01010101u * i) & 0x07070707u;
    }
    // the tile patterns: registers as the bulk warps of sweep_direct_kernel hold them
    uint32_t PLt[40], ltt[16], wt[8];
    if (PATTERN == PEAK_TILE_NEAR || PATTERN == PEAK_TILE_FAR) {
#pragma unroll
        for (int i = 0; i < 40; ++i) PLt[i] = seed * (i + 3) + tid;
#pragma unroll
        for (int i = 0; i < 16; ++i) ltt[i] = (seed + i * 0x01010101u) & 0x03030303u;
#pragma unroll
        for (int i = 0; i < 8; ++i) wt[i] = (seed * (i + 7) + tid) & 0x77777777u;
    }
    __syncthreads();
    const long long t0 = clock64();
    if (PATTERN == PEAK_TILE_NEAR || PATTERN == PEAK_TILE_FAR) {
        for (int it = 0; it < PEAK_TILE_ITERS; ++it) {
#pragma unroll
            for (int u = 0; u < 16; ++u) {
                const uint32_t sel = (u & 1) ? (wt[u >> 1] >> 16) : wt[u >> 1];
#pragma unroll
                for (int mm = 0; mm < 8; ++mm) {
                    uint32_t S;
                    asm volatile("prmt.b32 %0, %1, %2, %3;" : "=r"(S) : "r"(ltt[2 * mm]), "r"(ltt[2 * mm + 1]), "r"(sel));
                    const int tt = 7 - mm + 2 * u;
                    if (PATTERN == PEAK_TILE_NEAR) {
                        asm volatile("dp2a.lo.u32.u32 %0, %1, %2, %0;" : "+r"(acc[mm]) : "r"(PLt[tt]), "r"(S));
                        asm volatile("dp2a.hi.u32.u32 %0, %1, %2, %0;" : "+r"(acc[8 + mm]) : "r"(PLt[tt + 1]), "r"(S));
                    } else {
                        asm volatile("dp4a.u32.u32 %0, %1, %2, %0;" : "+r"(acc[8 * (u & 1) + mm]) : "r"(PLt[tt]), "r"(S));
                    }
                }
            }
            wt[it & 7] ^= acc[it & 7] & 0x77777777u;
        }
    } else
    for (int it = 0; it < PEAK_ITERS; ++it) {
#pragma unroll
        for (int i = 0; i < PEAK_UNROLL; ++i) {
            if (PATTERN == PEAK_IDP2A) {
                asm volatile("dp2a.lo.u32.u32 %0, %1, %2, %0;" : "+r"(acc[i]) : "r"(a[i]), "r"(b[i]));
            } else if (PATTERN == PEAK_IDP4A) {
                asm volatile("dp4a.u32.u32 %0, %1, %2, %0;" : "+r"(acc[i]) : "r"(a[i]), "r"(b[i]));
            } else if (PATTERN == PEAK_IMAD) {
                asm volatile("mad.lo.u32 %0, %1, %2, %0;" : "+r"(acc[i]) : "r"(a[i]), "r"(b[i]));
            } else if (PATTERN == PEAK_PRMT) {
                asm volatile("prmt.b32 %0, %1, %2, %0;" : "+r"(acc[i]) : "r"(a[i]), "r"(b[i]));
            } else if (PATTERN == PEAK_LOP3) {
                asm volatile("lop3.b32 %0, %1, %2, %0, 0x96;" : "+r"(acc[i]) : "r"(a[i]), "r"(b[i]));
            } else if (PATTERN == PEAK_MIX_BULK) {
                uint32_t S;
                asm volatile("prmt.b32 %0, %1, %2, %3;" : "=r"(S) : "r"(a[i]), "r"(acc[(i + 5) % PEAK_UNROLL]), "r"(b[i]));
                asm volatile("dp2a.lo.u32.u32 %0, %1, %2, %0;" : "+r"(acc[i]) : "r"(a[(i + 2) % PEAK_UNROLL]), "r"(S));
                asm volatile("dp2a.hi.u32.u32 %0, %1, %2, %0;" : "+r"(acc[(i + 8) % PEAK_UNROLL]) : "r"(a[(i + 3) % PEAK_UNROLL]), "r"(S));
            } else if (PATTERN == PEAK_MIX_BULK4) {
                uint32_t S;
                asm volatile("prmt.b32 %0, %1, %2, %3;" : "=r"(S) : "r"(a[i]), "r"(acc[(i + 5) % PEAK_UNROLL]), "r"(b[i]));
                asm volatile("dp2a.lo.u32.u32 %0, %1, %2, %0;" : "+r"(acc[i]) : "r"(a[(i + 2) % PEAK_UNROLL]), "r"(S));
                asm volatile("dp2a.hi.u32.u32 %0, %1, %2, %0;" : "+r"(acc[(i + 4) % PEAK_UNROLL]) : "r"(a[(i + 3) % PEAK_UNROLL]), "r"(S));
                asm volatile("dp2a.lo.u32.u32 %0, %1, %2, %0;" : "+r"(acc[(i + 8) % PEAK_UNROLL]) : "r"(a[(i + 5) % PEAK_UNROLL]), "r"(S));
                asm volatile("dp2a.hi.u32.u32 %0, %1, %2, %0;" : "+r"(acc[(i + 12) % PEAK_UNROLL]) : "r"(a[(i + 7) % PEAK_UNROLL]), "r"(S));
            } else if (PATTERN == PEAK_MIX_LOP) {
                uint32_t S;
                asm volatile("lop3.b32 %0, %1, %2, %3, 0x96;" : "=r"(S) : "r"(a[i]), "r"(acc[(i + 5) % PEAK_UNROLL]), "r"(b[i]));
                asm volatile("dp2a.lo.u32.u32 %0, %1, %2, %0;" : "+r"(acc[i]) : "r"(a[(i + 2) % PEAK_UNROLL]), "r"(S));
                asm volatile("dp2a.hi.u32.u32 %0, %1, %2, %0;" : "+r"(acc[(i + 8) % PEAK_UNROLL]) : "r"(a[(i + 3) % PEAK_UNROLL]), "r"(S));
            } else if (PATTERN == PEAK_MIX_MIRROR) {
                uint32_t S, S2, T;
                asm volatile("prmt.b32 %0, %1, %2, %3;" : "=r"(S) : "r"(a[i]), "r"(acc[(i + 5) % PEAK_UNROLL]), "r"(b[i]));
                asm volatile("prmt.b32 %0, %1, %2, %3;" : "=r"(S2) : "r"(a[i]), "r"(acc[(i + 6) % PEAK_UNROLL]), "r"(b[(i + 1) % PEAK_UNROLL]));
                asm volatile("add.u32 %0, %1, %2;" : "=r"(T) : "r"(S), "r"(S2));
                asm volatile("dp2a.lo.u32.u32 %0, %1, %2, %0;" : "+r"(acc[i]) : "r"(a[(i + 2) % PEAK_UNROLL]), "r"(T));
                asm volatile("dp2a.hi.u32.u32 %0, %1, %2, %0;" : "+r"(acc[(i + 8) % PEAK_UNROLL]) : "r"(a[(i + 3) % PEAK_UNROLL]), "r"(T));
            } else if (PATTERN == PEAK_LDS128) {
                uint4 v;
                const uint32_t addr = (uint32_t)__cvta_generic_to_shared(s_buf) + (uint32_t)(((tid + 32 * i) & 511) * 16);
                asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(addr));
                acc[i] += v.x ^ v.y ^ v.z ^ v.w;
            }
        }
    }
    const long long t1 = clock64();
    uint32_t r = 0;
#pragma unroll
    for (int i = 0; i < PEAK_UNROLL; ++i) r ^= acc[i];
    if (r == 0x12345u) sink[0] = r;   // never true in practice: keeps the chains alive
    __syncthreads();
    if (tid == 0) clocks[blockIdx.x] = t1 - t0;
}

// Counted warp-instructions per thread of one run of peak_kernel<PATTERN> (for the mixes: the IDP.2A only).
inline double peak_counted_ops(int pattern) {
    const double base = (double)PEAK_ITERS * PEAK_UNROLL;
    if (pattern == PEAK_MIX_BULK || pattern == PEAK_MIX_LOP || pattern == PEAK_MIX_MIRROR) return 2.0 * base;
    if (pattern == PEAK_MIX_BULK4) return 4.0 * base;
    if (pattern == PEAK_LDS128) return 16.0 * base;   // bytes per thread
    if (pattern == PEAK_TILE_NEAR) return 2.0 * 128.0 * PEAK_TILE_ITERS;
    if (pattern == PEAK_TILE_FAR) return 128.0 * PEAK_TILE_ITERS;
    return base;
}

typedef void (*peak_kernel_t)(long long*, uint32_t*, uint32_t);
inline peak_kernel_t peak_kernel_of(int pattern) {
    switch (pattern) {
        case PEAK_IDP2A: return peak_kernel<PEAK_IDP2A>;
        case PEAK_IDP4A: return peak_kernel<PEAK_IDP4A>;
        case PEAK_IMAD: return peak_kernel<PEAK_IMAD>;
        case PEAK_PRMT: return peak_kernel<PEAK_PRMT>;
        case PEAK_LOP3: return peak_kernel<PEAK_LOP3>;
        case PEAK_MIX_BULK: return peak_kernel<PEAK_MIX_BULK>;
        case PEAK_MIX_LOP: return peak_kernel<PEAK_MIX_LOP>;
        case PEAK_LDS128: return peak_kernel<PEAK_LDS128>;
        case PEAK_MIX_BULK4: return peak_kernel<PEAK_MIX_BULK4>;
        case PEAK_MIX_MIRROR: return peak_kernel<PEAK_MIX_MIRROR>;
        case PEAK_TILE_NEAR: return peak_kernel<PEAK_TILE_NEAR>;
        case PEAK_TILE_FAR: return peak_kernel<PEAK_TILE_FAR>;
        default: return nullptr;
    }
}

}  // namespace ptk

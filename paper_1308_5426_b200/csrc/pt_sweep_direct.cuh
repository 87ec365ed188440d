// pt_sweep_direct.cuh -- Metropolis sweep, direct-sum variant (PAPER.md:118-124:
// "compute only the energies corresponding to the flipped spin before and
// after", an O(L) sum per step, O(L^2) per sweep), organised for sm_100a.
//
// One CTA per replica, sites in blocks of 32 (site order 0..L-1, A5).
//
// BULK (all warps).  For the 32 sites i of a block, against the CURRENT spins,
//   S_i = sum_j Jq[(i-j) mod L] * s'_i(c_j),   s'_i(k) = 1 + [k==a_i] - [k==b_i],
// so that dE_i = S_i - sum_r Jq[r]  (Jq is symmetric, so (i-j) mod L indexes the
// same coupling as |i-j|; Jq[0] = 0 drops j == i).  The 32 x L pair terms of a
// block are split as 8 site groups (4 sites of equal parity) x L/64 ranges of
// 64 consecutive j, one (group, range) per thread.  The range is taken RELATIVE
// to the block start, so the 70 couplings a thread needs never change: they
// live in registers for the whole launch, as 16-bit halves packed in pairs
// (pt_kernels.cuh: pack_pairs_kernel).  Per 4 sites j the colour -> s' map is
// one PRMT (the packed 4-bit colours ARE the byte selectors of a per-site 8-byte
// table; hence q <= 8) and the multiply-accumulate is 4 IDP.2A (16-bit x 8-bit
// two-way dot products): 1.25 instructions per pair term, all integer, exact.
//
// CHAIN (warp 0, lane = site).  With dE_i valid at block start, the sequential
// acceptance of Eq. 8 inside the block only needs, for every
// accepted change f -> (a_f, b_f), the exact correction of the later lanes
//   dE_l += Jq[l-f] * ( [a_l==b_f] + [b_l==a_f] - [a_l==a_f] - [b_l==b_f] ),
// i.e. 32 unrolled steps of "is lane f accepted (ballot bit)? then correct and
// re-vote".  Integer arithmetic makes the result identical to the site-by-site
// order.  Proposals b_i and thresholds theta_i (reading A9) of all sites are
// drawn in parallel at the start of the sweep from the counter-based generator.
#pragma once
#include "pt_kernels.cuh"

namespace ptk {

constexpr int DIRECT_MAX_THREADS = 512;
constexpr int DIRECT_NPAIR = 35;  // packed coupling pairs per thread and half

__host__ __device__ inline bool direct_applies(int L, int q) {
    return (L % 64) == 0 && L >= 64 && L <= 64 * (DIRECT_MAX_THREADS / 8) && q <= 8;
}
__host__ __device__ inline int direct_threads(int L) {
    const int t = 8 * (L / 64);
    return t < 32 ? 32 : (t + 31) / 32 * 32;
}
// dynamic smem (32-bit words): theta[L] | lut[2L] | sp[W] | bq[W] | part[NW*32] | Jn[32]
__host__ __device__ inline size_t direct_smem_bytes(int L) {
    return (size_t)(3 * L + 2 * (L / 8) + (direct_threads(L) / 32) * 32 + 32) * 4;
}

__global__ void __launch_bounds__(DIRECT_MAX_THREADS, 1)
sweep_direct_kernel(Dev d, long long sweep0, int n_sweeps, int do_swap) {
    extern __shared__ uint32_t smem_d[];
    const int L = d.L, W = d.W, q = d.q;
    const int NT = blockDim.x, NW = NT >> 5;
    int32_t* theta = (int32_t*)smem_d;
    uint2* lut = (uint2*)(theta + L);
    uint32_t* sp = (uint32_t*)(lut + L);
    uint32_t* bq = sp + W;
    uint32_t* part = bq + W;
    int32_t* Jn = (int32_t*)(part + NW * 32);
    __shared__ int s_cnt[16];

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int e = blockIdx.x / d.n_rep, t = blockIdx.x % d.n_rep;
    const int st = d.perm[blockIdx.x];
    const size_t x = (size_t)e * d.n_rep + st;
    uint32_t* g_sp = d.spins + x * W;

    // thread -> (site group g, j-range jr); group g = sites 8(g>>1) + (g&1) + {0,2,4,6}
    const int g = tid & 7, jr = tid >> 3;
    const int par = g & 1, gbase = 8 * (g >> 1) + par;
    const bool active = jr < L / 64;

    // couplings of this thread: pair tt holds Jq[r], Jq[r-1] with r = R0 - 2 tt  (mod L)
    uint32_t PL[DIRECT_NPAIR], PH[DIRECT_NPAIR];
    {
        const int H = L / 2;
        const int R0 = ((gbase + 6 - 64 * jr) % L + L) % L;
        const uint32_t* lo = d.Jpair + (size_t)(2 * par) * H;
        const uint32_t* hi = lo + H;
#pragma unroll
        for (int tt = 0; tt < DIRECT_NPAIR; ++tt) {
            const int r = ((R0 - 2 * tt) % L + L) % L;
            const int m = (r - par) / 2;
            PL[tt] = active ? __ldg(lo + m) : 0u;
            PH[tt] = active ? __ldg(hi + m) : 0u;
        }
    }
    for (int w = tid; w < W; w += NT) sp[w] = g_sp[w];
    if (tid < 32) Jn[tid] = d.Jq[tid];
    // sum_r Jq[r]
    uint32_t rowsum;
    {
        uint32_t acc = 0;
        for (int r = lane; r < L; r += 32) acc += (uint32_t)d.Jq[r];
        rowsum = __reduce_add_sync(0xffffffffu, acc);
    }
    long long E = d.E[x];
    const double scale = d.thr_scale[t];
    const uint32_t c3 = ((uint32_t)(d.ens_base + e) << 4) | TAG_SWEEP;
    ObsAcc oa;
    __syncthreads();

    for (int s = 0; s < n_sweeps; ++s) {
        const uint32_t sweep = (uint32_t)(sweep0 + s + 1);
        // proposals, thresholds and colour tables of all sites (A6, A7, A9)
        for (int w = tid; w < W; w += NT) {
            const uint32_t word = sp[w];
            uint32_t bword = 0;
#pragma unroll
            for (int n = 0; n < 8; ++n) {
                const int i = 8 * w + n;
                const Philox4 p = philox4x32_10((uint32_t)i, sweep, (uint32_t)t, c3, d.key0, d.key1);
                const uint32_t a = (word >> (4 * n)) & 15u;
                const uint32_t k = __umulhi(p.w0, (uint32_t)(q - 1));
                const uint32_t b = k + (k >= a ? 1u : 0u);
                bword |= b << (4 * n);
                theta[i] = accept_threshold(uniform53(p.w1, p.w2), scale);
                const unsigned long long tab =
                    0x0101010101010101ull + (1ull << (8 * a)) - (1ull << (8 * b));  // byte k = s'(k)
                lut[i] = make_uint2((uint32_t)tab, (uint32_t)(tab >> 32));
            }
            bq[w] = bword;
        }
        __syncthreads();

        long long dE_acc = 0;  // warp 0: sum of accepted dE of this lane's sites
        int n_acc = 0;
        for (int i0 = 0; i0 < L; i0 += 32) {
            // ---- BULK ----
            uint32_t val[4] = {0u, 0u, 0u, 0u};
            if (active) {
                const int wj = ((i0 >> 3) + 8 * jr) % W;
                const int wj2 = (wj + 4) % W;
                const uint4 wa = *reinterpret_cast<const uint4*>(sp + wj);
                const uint4 wb = *reinterpret_cast<const uint4*>(sp + wj2);
                const uint32_t words[8] = {wa.x, wa.y, wa.z, wa.w, wb.x, wb.y, wb.z, wb.w};
                uint2 lt[4];
                uint32_t alo[4] = {0u, 0u, 0u, 0u}, ahi[4] = {0u, 0u, 0u, 0u};
#pragma unroll
                for (int m = 0; m < 4; ++m) lt[m] = lut[i0 + gbase + 2 * m];
#pragma unroll
                for (int u = 0; u < 16; ++u) {
                    const uint32_t sel = (u & 1) ? (words[u >> 1] >> 16) : words[u >> 1];
#pragma unroll
                    for (int m = 0; m < 4; ++m) {
                        const uint32_t S = __byte_perm(lt[m].x, lt[m].y, sel);
                        const int tt = 3 - m + 2 * u;
                        alo[m] = __dp2a_lo(PL[tt], S, alo[m]);
                        alo[m] = __dp2a_hi(PL[tt + 1], S, alo[m]);
                        ahi[m] = __dp2a_lo(PH[tt], S, ahi[m]);
                        ahi[m] = __dp2a_hi(PH[tt + 1], S, ahi[m]);
                    }
                }
#pragma unroll
                for (int m = 0; m < 4; ++m) val[m] = alo[m] + (ahi[m] << 16);
            }
#pragma unroll
            for (int m = 0; m < 4; ++m) {
                val[m] += __shfl_xor_sync(0xffffffffu, val[m], 8);
                val[m] += __shfl_xor_sync(0xffffffffu, val[m], 16);
            }
            if (lane < 8) {
#pragma unroll
                for (int m = 0; m < 4; ++m) part[warp * 32 + gbase + 2 * m] = val[m];
            }
            __syncthreads();

            // ---- CHAIN ----
            if (warp == 0) {
                uint32_t S = 0;
                for (int w = 0; w < NW; ++w) S += part[w * 32 + lane];
                int dE = (int)(S - rowsum);
                const int th = theta[i0 + lane];
                uint32_t aw[4], bw[4];
#pragma unroll
                for (int k = 0; k < 4; ++k) { aw[k] = sp[(i0 >> 3) + k]; bw[k] = bq[(i0 >> 3) + k]; }
                const int a = (int)((aw[lane >> 3] >> ((lane & 7) << 2)) & 15u);
                const int b = (int)((bw[lane >> 3] >> ((lane & 7) << 2)) & 15u);
                int Jd[32];
#pragma unroll
                for (int f = 0; f < 32; ++f) Jd[f] = Jn[lane > f ? lane - f : 0];  // Jn[0] = 0: lanes <= f unchanged
                unsigned mask = __ballot_sync(0xffffffffu, dE <= th);
#pragma unroll
                for (int f = 0; f < 32; ++f) {
                    if ((mask >> f) & 1u) {  // lane f's decision is final: accepted
                        const int af = (int)((aw[f >> 3] >> ((f & 7) << 2)) & 15u);
                        const int bf = (int)((bw[f >> 3] >> ((f & 7) << 2)) & 15u);
                        const int coef = (a == bf) + (b == af) - (a == af) - (b == bf);
                        dE += Jd[f] * coef;
                        mask = __ballot_sync(0xffffffffu, dE <= th);
                    }
                }
                const bool acc = (mask >> lane) & 1u;
                if (acc) dE_acc += dE;
                n_acc += acc ? 1 : 0;
                const uint32_t nv = (uint32_t)(acc ? b : a) << ((lane & 7) << 2);
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    const uint32_t wk = __reduce_or_sync(0xffffffffu, (lane >> 3) == k ? nv : 0u);
                    if (lane == k) sp[(i0 >> 3) + k] = wk;
                }
            }
            __syncthreads();
        }
        if (warp == 0) {
            for (int o = 16; o > 0; o >>= 1) {
                dE_acc += __shfl_xor_sync(0xffffffffu, dE_acc, o);
                n_acc += __shfl_xor_sync(0xffffffffu, n_acc, o);
            }
            E += dE_acc;
            oa.acc += n_acc;
        }
        // a8: sample after the sweep, before the swap event (A15)
        const int nmax = count_nmax(sp, W, q, s_cnt);
        if (tid == 0) { oa.att += L; oa.sample(E, nmax); }
        __syncthreads();
    }

    for (int w = tid; w < W; w += NT) g_sp[w] = sp[w];
    if (tid == 0) { d.E[x] = E; oa.flush(d.obs + blockIdx.x); }
    if (do_swap) arrive_and_swap(d, e, (uint32_t)(sweep0 + n_sweeps));
}

// Returns a cudaError_t as int.
inline int launch_sweep_direct(const Dev& d, long long sweep0, int n_sweeps, int do_swap, cudaStream_t stream) {
    const size_t smem = direct_smem_bytes(d.L);
    cudaError_t err = cudaFuncSetAttribute(sweep_direct_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (err != cudaSuccess) return (int)err;
    sweep_direct_kernel<<<d.n_ens * d.n_rep, direct_threads(d.L), smem, stream>>>(d, sweep0, n_sweeps, do_swap);
    return (int)cudaGetLastError();
}

}  // namespace ptk

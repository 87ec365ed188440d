// pt_sweep_direct.cuh -- Metropolis sweep, direct-sum variant (PAPER.md:118-124:
// "compute only the energies corresponding to the flipped spin before and
// after", an O(L) sum per step, O(L^2) per sweep), organised for sm_100a.
//
// One CTA per replica, sites in blocks of 32 (site order 0..L-1, A5).  Warps are
// specialised and the two halves of a block's work run CONCURRENTLY on
// consecutive blocks: in interval k (between two CTA barriers)
//   * the BULK warps sum block k+1 against the spins as they are, and
//   * one CHAIN warp takes the sequential accept/reject decisions of block k,
//     while the other chain warp prepares block k+1.
//
// BULK (NTB = L/8 threads).  For the 32 sites i of a block,
//   S_i = sum_j Jq[(i-j) mod L] * s'_i(c_j),   s'_i(k) = 1 + [k==a_i] - [k==b_i],
// so that dE_i = S_i - sum_r Jq[r]  (Jq is symmetric, so (i-j) mod L indexes the
// same coupling as |i-j|; Jq[0] = 0 drops j == i).  The 32 x L pair terms of a
// block are split as 8 site groups (4 sites of equal parity) x L/64 ranges of
// 64 consecutive j, one (group, range) per thread.  The range is taken RELATIVE
// to the block start, so the 70 couplings a thread needs never change: they
// live in registers for the whole launch as 16-bit halves packed in pairs
// (pt_kernels.cuh: pack_pairs_kernel).  Per 4 sites j the colour -> s' map is
// one PRMT (the packed 4-bit colours ARE the byte selectors of a per-site 8-byte
// table; hence q <= 8) and the multiply-accumulate is IDP.2A (16-bit x 8-bit
// two-way dot products), all integer, exact.  The HIGH halves Jq[r] >> 16 are
// non-zero only for r <= r_hi (71 at L=4096, sigma=0.3): with FULL_HI = false
// the bulk warps sum the low halves only (0.5 IDP.2A per pair term) and the
// high halves of the 224 sites around the block are summed by the preparing
// chain warp (NEAR); FULL_HI = true keeps both halves in the bulk warps (small
// L or small sigma, where r_hi is not small).
//
// Because block k+1 is summed while block k is still being decided, the bulk
// reads block k as it was at the START of the sweep (sp0) and everything else
// live (sp): blocks < k are final, blocks > k untouched.  The chain warp then
// corrects for the changes accepted in block k exactly like for those inside
// its own block:
//
// CHAIN (lane = site).  With dE_l valid for the stale configuration, the
// sequential acceptance of Eq. 8 needs, for every accepted
// change f: a_f -> b_f at an earlier site, the exact correction
//   dE_l += Jq[l-f] * ( s'_l(b_f) - s'_l(a_f) ),
// 32 predicated adds for the previous block (all known at once) and 32
// dependent steps "vote on lane f, add its correction" inside the block.  The
// 64 correction terms of a lane are computed ahead of time (PREP) while the
// other chain warp is deciding the previous block.  Integer arithmetic makes
// the result identical to the site-by-site order.  Proposals b_i and
// thresholds theta_i (reading A9) of all sites are drawn in parallel at the
// start of the sweep from the counter-based generator.
#pragma once
#include "pt_kernels.cuh"

namespace ptk {

constexpr int DIRECT_MAX_BULK = 512;
constexpr int DIRECT_MAX_THREADS = DIRECT_MAX_BULK + 64;  // + two chain warps
constexpr int DIRECT_NPAIR = 35;   // packed coupling pairs per thread and half
constexpr int DIRECT_NEAR_R = 95;  // NEAR covers |i-j| <= 95: 224 sites around a block

__host__ __device__ inline bool direct_applies(int L, int q) {
    return (L % 64) == 0 && L >= 64 && L <= 64 * (DIRECT_MAX_BULK / 8) && q <= 8;
}
__host__ __device__ inline int direct_bulk_threads(int L) {
    const int t = 8 * (L / 64);
    return t < 32 ? 32 : (t + 31) / 32 * 32;
}
__host__ __device__ inline int direct_threads(int L) { return direct_bulk_threads(L) + 64; }
// dynamic smem (32-bit words): theta[L] | lut[2L] | sp[W] | sp0[W] | bq[W] | part[64] | Jz[96] | PPhi[256]
__host__ __device__ inline size_t direct_smem_bytes(int L) {
    return (size_t)(3 * L + 3 * (L / 8) + 64 + 96 + 256) * 4;
}

__device__ __forceinline__ int dp4a_s32_u32(int a, uint32_t b, int c) {
    int d;
    asm("dp4a.s32.u32 %0, %1, %2, %3;" : "=r"(d) : "r"(a), "r"(b), "r"(c));
    return d;
}

// 8 accept bits -> 8 nibbles of 0xF
__device__ __forceinline__ uint32_t expand_bits_to_nibbles(uint32_t m8) {
    uint32_t x = m8 & 0xffu;
    x = (x | (x << 12)) & 0x000F000Fu;
    x = (x | (x << 6)) & 0x03030303u;
    x = (x | (x << 3)) & 0x11111111u;
    return x * 15u;
}

// CTA-wide barrier usable from role-specialised code paths (every warp executes the same number of them).
__device__ __forceinline__ void cta_sync() { asm volatile("bar.sync 0;" ::: "memory"); }

struct DirectSmem {
    int32_t* theta;   // [L]  acceptance thresholds of the running sweep
    uint2* lut;       // [L]  per-site colour -> s' byte table
    uint32_t* sp;     // [W]  live packed spins
    uint32_t* sp0;    // [W]  spins at the start of the running sweep
    uint32_t* bq;     // [W]  proposed colours
    uint32_t* part;   // [2][32] block sums S_i, double buffered
    int32_t* Jz;      // [96] Jz[n] = 0 for n < 32, Jq[n - 32] above
    uint32_t* PPhi;   // [256] index r + 128 -> hi(|r|) | hi(|r-1|) << 16, hi(d) = Jq[d] >> 16 for 1 <= d <= r_hi
};

// Start of a sweep, all threads: proposals, thresholds and colour tables of all sites (A6, A7, A9) and the
// snapshot of the spins.
__device__ __forceinline__ void direct_draw(const Dev& d, const DirectSmem& m, uint32_t sweep, int t, uint32_t c3,
                                            double scale) {
    const int W = d.W, q = d.q;
    for (int w = threadIdx.x; w < W; w += blockDim.x) {
        const uint32_t word = m.sp[w];
        uint32_t bword = 0;
#pragma unroll
        for (int n = 0; n < 8; ++n) {
            const int i = 8 * w + n;
            const Philox4 p = philox4x32_10((uint32_t)i, sweep, (uint32_t)t, c3, d.key0, d.key1);
            const uint32_t a = (word >> (4 * n)) & 15u;
            const uint32_t k = __umulhi(p.w0, (uint32_t)(q - 1));
            const uint32_t b = k + (k >= a ? 1u : 0u);
            bword |= b << (4 * n);
            m.theta[i] = accept_threshold(uniform53(p.w1, p.w2), scale);
            const unsigned long long tab =
                0x0101010101010101ull + (1ull << (8 * a)) - (1ull << (8 * b));  // byte k = s'(k)
            m.lut[i] = make_uint2((uint32_t)tab, (uint32_t)(tab >> 32));
        }
        m.bq[w] = bword;
        m.sp0[w] = word;
    }
}

// N_max of the configuration (Eq. 10), as count_nmax but on cta_sync.
__device__ __forceinline__ int direct_nmax(const uint32_t* sp, int W, int q, int* s_cnt) {
    if (threadIdx.x < 16) s_cnt[threadIdx.x] = 0;
    cta_sync();
    for (int w = threadIdx.x; w < W; w += blockDim.x) {
        const uint32_t word = sp[w];
        for (int k = 0; k < q; ++k) {
            const int c = __popc(match_nibbles(word, (uint32_t)k));
            if (c) atomicAdd(&s_cnt[k], c);
        }
    }
    cta_sync();
    int nmax = 0;
    if (threadIdx.x == 0)
        for (int k = 0; k < q; ++k) nmax = max(nmax, s_cnt[k]);
    return nmax;
}

template <bool FULL_HI>
__global__ void __launch_bounds__(DIRECT_MAX_THREADS, 1)
sweep_direct_kernel(Dev d, long long sweep0, int n_sweeps, int do_swap, int r_hi) {
    extern __shared__ uint32_t smem_d[];
    const int L = d.L, W = d.W, q = d.q;
    const int NT = blockDim.x, NTB = NT - 64;
    const int NB = L >> 5;
    DirectSmem m;
    m.theta = (int32_t*)smem_d;
    m.lut = (uint2*)(m.theta + L);
    m.sp = (uint32_t*)(m.lut + L);
    m.sp0 = m.sp + W;
    m.bq = m.sp0 + W;
    m.part = m.bq + W;
    m.Jz = (int32_t*)(m.part + 64);
    m.PPhi = (uint32_t*)(m.Jz + 96);
    __shared__ int s_cnt[16];
    __shared__ uint32_t s_mask[2];
    __shared__ long long s_dE[2];
    __shared__ int s_nacc[2];

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int e = blockIdx.x / d.n_rep, t = blockIdx.x % d.n_rep;
    const int st = d.perm[blockIdx.x];
    const size_t x = (size_t)e * d.n_rep + st;
    uint32_t* g_sp = d.spins + x * W;

    for (int w = tid; w < W; w += NT) m.sp[w] = g_sp[w];
    if (tid < 96) m.Jz[tid] = tid < 32 ? 0 : d.Jq[tid - 32];
    for (int n = tid; n < 256; n += NT) {
        const int r = n - 128;
        const int r0 = r < 0 ? -r : r, r1 = r - 1 < 0 ? 1 - r : r - 1;
        const uint32_t h0 = (r0 >= 1 && r0 <= r_hi) ? ((uint32_t)d.Jq[r0] >> 16) : 0u;
        const uint32_t h1 = (r1 >= 1 && r1 <= r_hi) ? ((uint32_t)d.Jq[r1] >> 16) : 0u;
        m.PPhi[n] = h0 | (h1 << 16);
    }
    if (tid < 64) m.part[tid] = 0u;
    const double scale = d.thr_scale[t];
    const uint32_t c3 = ((uint32_t)(d.ens_base + e) << 4) | TAG_SWEEP;

    if (tid < NTB) {
        // =========================== BULK warps ===========================
        // thread -> (site group g, j-range jr); group g = sites 8(g>>1) + (g&1) + {0,2,4,6}
        const int g = tid & 7, jr = tid >> 3;
        const int par = g & 1, gbase = 8 * (g >> 1) + par;
        const int NJR = L / 64;
        const bool active = jr < NJR;
        // couplings of this thread: pair tt holds Jq[r], Jq[r-1] with r = R0 - 2 tt  (mod L)
        uint32_t PL[DIRECT_NPAIR];
        uint32_t PH[FULL_HI ? DIRECT_NPAIR : 1];
        {
            const int H = L / 2;
            const int R0 = ((gbase + 6 - 64 * jr) % L + L) % L;
            const uint32_t* lo = d.Jpair + (size_t)(2 * par) * H;
            const uint32_t* hi = lo + H;
#pragma unroll
            for (int tt = 0; tt < DIRECT_NPAIR; ++tt) {
                const int r = ((R0 - 2 * tt) % L + L) % L;
                const int mm = (r - par) / 2;
                PL[tt] = active ? __ldg(lo + mm) : 0u;
                if (FULL_HI) PH[tt] = active ? __ldg(hi + mm) : 0u;
            }
            if (!FULL_HI) PH[0] = 0u;
        }
        long long E = d.E[x];
        ObsAcc oa;
        cta_sync();

        for (int s = 0; s < n_sweeps; ++s) {
            direct_draw(d, m, (uint32_t)(sweep0 + s + 1), t, c3, scale);
            cta_sync();
            for (int kb = 0; kb <= NB; ++kb) {   // interval kb-1: sum block kb
                if (kb < NB) {
                    const int i0 = kb << 5;
                    uint32_t val[4] = {0u, 0u, 0u, 0u};
                    if (active) {
                        const int wj = ((i0 >> 3) + 8 * jr) % W;
                        const int wj2 = (wj + 4) % W;
                        const uint4 wa = *reinterpret_cast<const uint4*>(m.sp + wj);
                        // the second half of the last range is block kb-1, which is being decided: sweep-start copy
                        const uint4 wb = *reinterpret_cast<const uint4*>((jr == NJR - 1 ? m.sp0 : m.sp) + wj2);
                        const uint32_t words[8] = {wa.x, wa.y, wa.z, wa.w, wb.x, wb.y, wb.z, wb.w};
                        uint2 lt[4];
                        uint32_t alo[4] = {0u, 0u, 0u, 0u}, ahi[4] = {0u, 0u, 0u, 0u};
#pragma unroll
                        for (int mm = 0; mm < 4; ++mm) lt[mm] = m.lut[i0 + gbase + 2 * mm];
#pragma unroll
                        for (int u = 0; u < 16; ++u) {
                            const uint32_t sel = (u & 1) ? (words[u >> 1] >> 16) : words[u >> 1];
#pragma unroll
                            for (int mm = 0; mm < 4; ++mm) {
                                const uint32_t S = __byte_perm(lt[mm].x, lt[mm].y, sel);
                                const int tt = 3 - mm + 2 * u;
                                alo[mm] = __dp2a_lo(PL[tt], S, alo[mm]);
                                alo[mm] = __dp2a_hi(PL[tt + 1], S, alo[mm]);
                                if (FULL_HI) {
                                    ahi[mm] = __dp2a_lo(PH[FULL_HI ? tt : 0], S, ahi[mm]);
                                    ahi[mm] = __dp2a_hi(PH[FULL_HI ? tt + 1 : 0], S, ahi[mm]);
                                }
                            }
                        }
#pragma unroll
                        for (int mm = 0; mm < 4; ++mm) val[mm] = alo[mm] + (ahi[mm] << 16);
                    }
#pragma unroll
                    for (int mm = 0; mm < 4; ++mm) {
                        val[mm] += __shfl_xor_sync(0xffffffffu, val[mm], 8);
                        val[mm] += __shfl_xor_sync(0xffffffffu, val[mm], 16);
                    }
                    if (lane < 8) {
#pragma unroll
                        for (int mm = 0; mm < 4; ++mm) atomicAdd(&m.part[(kb & 1) * 32 + gbase + 2 * mm], val[mm]);
                    }
                }
                cta_sync();
            }
            cta_sync();  // chain warps have published their sums
            // a8: sample after the sweep, before the swap event (A15)
            const int nmax = direct_nmax(m.sp, W, q, s_cnt);
            if (tid == 0) {
                E += s_dE[0] + s_dE[1];
                oa.acc += s_nacc[0] + s_nacc[1];
                oa.att += L;
                oa.sample(E, nmax);
            }
            cta_sync();
        }
        if (tid == 0) { d.E[x] = E; oa.flush(d.obs + blockIdx.x); }
    } else {
        // =========================== CHAIN warps ===========================
        const int cw = warp - (NTB >> 5);  // chain warp 0 decides the even blocks, 1 the odd blocks
        // sum_r Jq[r]
        uint32_t rowsum;
        {
            uint32_t acc = 0;
            for (int r = lane; r < L; r += 32) acc += (uint32_t)d.Jq[r];
            rowsum = __reduce_add_sync(0xffffffffu, acc);
        }
        cta_sync();

        for (int s = 0; s < n_sweeps; ++s) {
            direct_draw(d, m, (uint32_t)(sweep0 + s + 1), t, c3, scale);
            cta_sync();
            // state carried from PREP (interval k-1) to CHAIN (interval k)
            int cin[32], cpv[32];
            int th = 0;
            long long dE_acc = 0;
            int n_acc = 0;
#pragma unroll
            for (int f = 0; f < 32; ++f) { cin[f] = 0; cpv[f] = 0; }

            for (int k = -1; k < NB; ++k) {
                if (k >= 0 && (k & 1) == cw) {
                    // ---- CHAIN of block k ----
                    const int i0 = k << 5;
                    const uint32_t S = m.part[(k & 1) * 32 + lane];
                    m.part[(k & 1) * 32 + lane] = 0u;
                    int dE = (int)(S - rowsum);
                    const uint32_t mp = k > 0 ? s_mask[(k - 1) & 1] : 0u;
                    {
                        int c0 = 0, c1 = 0, c2 = 0, c3s = 0;
#pragma unroll
                        for (int f = 0; f < 32; f += 4) {
                            c0 += ((mp >> f) & 1u) ? cpv[f] : 0;
                            c1 += ((mp >> (f + 1)) & 1u) ? cpv[f + 1] : 0;
                            c2 += ((mp >> (f + 2)) & 1u) ? cpv[f + 2] : 0;
                            c3s += ((mp >> (f + 3)) & 1u) ? cpv[f + 3] : 0;
                        }
                        dE += (c0 + c1) + (c2 + c3s);
                    }
                    unsigned mask = __ballot_sync(0xffffffffu, dE <= th);
#pragma unroll
                    for (int f = 0; f < 31; ++f) {
                        dE += ((mask >> f) & 1u) ? cin[f] : 0;  // cin[f] = 0 for lanes <= f: their decision is final
                        mask = __ballot_sync(0xffffffffu, dE <= th);
                    }
                    if ((mask >> lane) & 1u) dE_acc += dE;
                    if (lane == 0) { n_acc += __popc(mask); s_mask[k & 1] = mask; }
                    if (lane < 4) {
                        const int w = (i0 >> 3) + lane;
                        const uint32_t nm = expand_bits_to_nibbles(mask >> (8 * lane));
                        m.sp[w] = (m.sp[w] & ~nm) | (m.bq[w] & nm);
                    }
                } else if (k + 1 < NB && ((k + 1) & 1) == cw) {
                    // ---- PREP of block k+1: threshold and correction terms; NEAR: high halves around the block ----
                    const int i0 = (k + 1) << 5;
                    const int il = i0 + lane;
                    const int ip = (il - 32 + L) % L;
                    th = m.theta[il];
                    const uint2 tab = m.lut[il];
                    const uint32_t sel = (uint32_t)get_nibble(m.sp, il) | ((uint32_t)get_nibble(m.bq, il) << 4);
                    const uint32_t selp = (uint32_t)get_nibble(m.sp0, ip) | ((uint32_t)get_nibble(m.bq, ip) << 4);
                    const int32_t* Jl = m.Jz + 32 + lane;
#pragma unroll
                    for (int f = 0; f < 32; ++f) {
                        const uint32_t sf = __shfl_sync(0xffffffffu, sel, f);
                        const uint32_t sv = __byte_perm(tab.x, tab.y, sf);  // byte 0 = s'_l(a_f), byte 1 = s'_l(b_f)
                        cin[f] = Jl[-f] * dp4a_s32_u32(0x000001ff, sv, 0);
                        const uint32_t pf = __shfl_sync(0xffffffffu, selp, f);
                        const uint32_t pv = __byte_perm(tab.x, tab.y, pf);
                        cpv[f] = Jl[32 - f] * dp4a_s32_u32(0x000001ff, pv, 0);
                    }
                    if (!FULL_HI) {
                        uint32_t acc = 0;
                        const int w0 = (i0 >> 3) - 12 + W;   // window: sites i0-96 .. i0+127 = 28 words
                        const uint32_t* pp = m.PPhi + 128 + lane + 96;
#pragma unroll 4
                        for (int n = 0; n < 28; ++n) {
                            const int w = (w0 + n) % W;
                            // words 8..11 of the window are block k (being decided): sweep-start copy
                            const uint32_t word = (n >= 8 && n < 12) ? m.sp0[w] : m.sp[w];
                            const uint32_t S0 = __byte_perm(tab.x, tab.y, word);
                            const uint32_t S1 = __byte_perm(tab.x, tab.y, word >> 16);
                            // site j = i0 - 96 + 8n + {0..7}; r = il - j = lane + 96 - 8n - {0..7}
                            acc = __dp2a_lo(pp[-8 * n], S0, acc);
                            acc = __dp2a_hi(pp[-8 * n - 2], S0, acc);
                            acc = __dp2a_lo(pp[-8 * n - 4], S1, acc);
                            acc = __dp2a_hi(pp[-8 * n - 6], S1, acc);
                        }
                        atomicAdd(&m.part[((k + 1) & 1) * 32 + lane], acc << 16);
                    }
                }
                cta_sync();
            }
            for (int o = 16; o > 0; o >>= 1) dE_acc += __shfl_xor_sync(0xffffffffu, dE_acc, o);
            if (lane == 0) { s_dE[cw] = dE_acc; s_nacc[cw] = n_acc; }
            cta_sync();
            direct_nmax(m.sp, W, q, s_cnt);
            cta_sync();
        }
    }

    cta_sync();
    for (int w = tid; w < W; w += NT) g_sp[w] = m.sp[w];
    if (do_swap) arrive_and_swap(d, e, (uint32_t)(sweep0 + n_sweeps));
}

// Returns a cudaError_t as int.  r_hi = largest r <= L/2 with Jq[r] >= 2^16 (0 if none).
inline int launch_sweep_direct(const Dev& d, long long sweep0, int n_sweeps, int do_swap, int r_hi,
                               cudaStream_t stream) {
    const size_t smem = direct_smem_bytes(d.L);
    const bool full_hi = r_hi > DIRECT_NEAR_R || d.L < 256;  // NEAR's 224-site window must not wrap onto itself
    auto kern = full_hi ? sweep_direct_kernel<true> : sweep_direct_kernel<false>;
    cudaError_t err = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (err != cudaSuccess) return (int)err;
    kern<<<d.n_ens * d.n_rep, direct_threads(d.L), smem, stream>>>(d, sweep0, n_sweeps, do_swap, r_hi);
    return (int)cudaGetLastError();
}

}  // namespace ptk

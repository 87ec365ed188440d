// pt_sweep_direct.cuh -- Metropolis sweep, direct-sum variant (PAPER.md:118-124:
// "compute only the energies corresponding to the flipped spin before and
// after", an O(L) sum per step, O(L^2) per sweep), organised for sm_100a.
//
// One CTA per replica, sites in blocks of 32 (site order 0..L-1, A5).  Warps are
// specialised: NTB = 4*(L/64) threads of BULK warps (8 warps at L=4096) and four
// CHAIN warps (one per SM sub-partition), coupled only through two pairs of shared-memory mbarriers, so
// that the bulk sum of block k+1 runs while block k is being decided.
//
// DRAW (all threads, once per sweep).  Proposals b_i, integer thresholds
// theta_i (reading A9) and the per-site colour tables of all sites are drawn in
// parallel from the counter-based generator; sp0 keeps the spins as they are
// at the start of the sweep.
//
// BULK.  For the 32 sites i of a block,
//   S_i = sum_j Jq[(i-j) mod L] * s'_i(c_j),   s'_i(k) = 1 + [k==a_i] - [k==b_i],
// so that dE_i = S_i - sum_r Jq[r]  (Jq is symmetric, so (i-j) mod L indexes the
// same coupling as |i-j|; Jq[0] = 0 drops j == i).  The 32 x L pair terms of a
// block are split as 4 site groups (the 8 sites of equal parity of a 16-site
// half) x L/64 ranges of 64 consecutive j, one (group, range) per thread: a fat
// tile (up to 168 registers, one CTA per SM; the MINB=2 build of the same code
// fits 80 registers for persistent launches that need more CTAs per SM), so
// that every unpacked word of colours serves 8 sites.  The range is taken RELATIVE
// to the block start, so the couplings a thread needs never change: they live
// in registers for the whole launch as 16-bit halves packed in pairs
// (pt_kernels.cuh: pack_pairs_kernel).  Per 4 sites j the colour -> s' map is
// one PRMT (the packed 4-bit colours ARE the byte selectors of a per-site 8-byte
// table; hence q <= 8) and the multiply-accumulate is IDP.2A (16-bit x 8-bit
// two-way dot products), all integer, exact.  The HIGH halves Jq[r] >> 16 are
// non-zero only for r <= r_hi (71 at L=4096, sigma=0.3): with NEARQ != 0 the
// main loop sums the low halves only (0.5 IDP.2A per pair term) and each thread
// adds the high halves of NEARQ of the quads of sites within distance off - 1
// of the block (NEAR; off = 96, 160, .., 352, the smallest above r_hi: 56, 88, ..,
// 184 quads); NEARQ = 0 keeps both halves everywhere (rings shorter than 2 off + 64).
// Block sums: a transpose-shuffle reduction leaves one site's partial sum per
// lane, then one shared-memory atomic per lane; every bulk warp then arrives on
// full[k&1].  Before block k a bulk warp waits on
// done[k&1] (block k-2 decided), so it reads: blocks < k-1 final, block k-1 as
// it was at the START of the sweep (sp0; it may still be changing), blocks >= k
// untouched.
//
// CHAIN (lane = site l, every chain warp holds all 32 slacks y_l = theta_l - dE_l).
// For an accepted change a_f -> b_f at an earlier site f, dE_l changes by
//   cm[f][l] = Jq[l-f] * ( s'_l(b_f) - s'_l(a_f) )          (exact, integer).
// Chain warp cw computes the rows f = 8cw..8cw+7 of the previous block (whose
// changes the bulk did not see) and of the own block from registers (CORR:
// PRMT + IDP.4A + IMAD per entry, before it waits on full[k&1]).  The accept
// mask a of the block is the unique solution of the triangular system
//   a_l = [ y_l - sum_{f<l} a_f cm[f][l] >= 0 ],
// which the site-by-site order of Eq. 8 solves by forward
// substitution.  Here it is solved by fixed-point rounds a <- F(a) starting
// from "no correction": after t rounds the first t bits are exact, so at most
// 32 rounds give exactly the sequential result; measured: 2.8 rounds per block
// for the hottest replica of configs[3], 0-1 for cold ones.  A round is a masked
// sum of 8 rows per warp (LOP3 -> predicate, SEL, IADD3: ALU pipe only, the FMA
// pipe is saturated by BULK), an exchange of the four partial sums through
// shared memory (named barrier 1) and a ballot.  Chain warp 0 writes the new
// spins; after the block's closing named barrier (all chain warps have read the
// block sums by then, also when the block needed no round) it clears the sums
// for block k+2 and arrives on done[k&1].  Integer arithmetic makes all of this
// independent of the order of summation (parity tests: bit-identical).
//
// OBSERVABLES, SWAPS.  Lane 0 of chain warp 0 owns the configuration's running
// energy and the slot's accumulators (shared memory); it samples them after
// every sweep (A15).  swap_mode 1: the launch ends with one swap event, run by
// the CTA that arrives last (nobody waits).  swap_mode 2 (persistent,
// cooperative launch, all replicas co-resident): the launch runs many sweeps;
// at a swap event every CTA publishes its energy, meets the others at a counter
// barrier in global memory, and evaluates the whole event on its own copy of the
// slot -> storage permutation (direct_swap_in_kernel); the configuration keeps
// its CTA and shared memory, the temperature, RNG slot and accumulators move.
#pragma once
#include "pt_kernels.cuh"

namespace ptk {

constexpr int DIRECT_SITES = 8;     // sites of a block per bulk thread (4 threads x 8 sites = 32)
constexpr int DIRECT_MAX_BULK = 256;
constexpr int DIRECT_CHAIN_WARPS = 4;                       // one per SM sub-partition
constexpr int DIRECT_MAX_THREADS = DIRECT_MAX_BULK + 32 * DIRECT_CHAIN_WARPS;
// L > 4096 (the paper's benchmark range reaches L = 10240): more j-ranges, hence more bulk threads, with
// the 80-register build of the same code (768 threads x 80 registers fill the register file of an SM).
constexpr int DIRECT_BIG_BULK = 640;
// 1024 < L <= 2048: 128 bulk + 128 chain threads; two such CTAs per SM with 128 registers per thread
constexpr int DIRECT_MID_THREADS = 256;
constexpr int DIRECT_BIG_THREADS = DIRECT_BIG_BULK + 32 * DIRECT_CHAIN_WARPS;
constexpr int DIRECT_STATIC_SMEM = 14 * 1024;   // upper bound of the sweep kernel's static shared memory (13568 B)
constexpr int DIRECT_NPAIR = 39;   // packed coupling pairs per thread and half: 64 + 2*7 couplings
constexpr int ENERGY_MAX_THREADS = 512, ENERGY_NPAIR = 35;   // energy_direct_kernel: 4 sites x 64 j per thread
// NEAR covers |i-j| < off, off = 96, 160, .., 352 (the smallest that is > r_hi): the off/2 + 8 quads of sites from
// off sites before the block to off sites behind it (56 quads for off = 96: r_hi = 71 at L = 4096, sigma = 0.3; 88
// for 160: sigma = 0.2; 184 for 352: r_hi = 337 at L = 4096, sigma = 0.1 -- the periodic images add to every coupling,
// so r_hi grows as the ring shrinks).  0: r_hi is beyond every window.
__host__ __device__ inline int direct_near_off(int r_hi) {
    return r_hi < 96 ? 96 : r_hi < 160 ? 160 : r_hi < 224 ? 224 : r_hi < 288 ? 288 : r_hi < 352 ? 352 : 0;
}
constexpr int DIRECT_MAX_PERSIST_REP = 512;   // replicas per ensemble in a persistent launch (static shared arrays)

__host__ __device__ inline size_t direct_smem_bytes(int L, int q);
__host__ __device__ inline bool direct_applies(int L, int q) {
    return (L % 64) == 0 && L >= 64 && L <= 64 * (DIRECT_BIG_BULK / 4) && q <= 16 &&
           direct_smem_bytes(L, q) + DIRECT_STATIC_SMEM <= 227 * 1024;
}
// energy_direct_kernel keeps one j-range per thread of a single CTA: L <= 4096 (beyond: the plain energy_kernel)
__host__ __device__ inline bool energy_direct_applies(int L, int q) {
    return direct_applies(L, q) && L <= 64 * (ENERGY_MAX_THREADS / 8);
}
__host__ __device__ inline int direct_bulk_threads(int L) {
    const int t = 4 * (L / 64);
    return t < 32 ? 32 : (t + 31) / 32 * 32;
}
__host__ __device__ inline int energy_threads(int L) {
    const int t = 8 * (L / 64);
    return t < 32 ? 32 : (t + 31) / 32 * 32;
}
__host__ __device__ inline int direct_threads(int L, int cw = DIRECT_CHAIN_WARPS) { return direct_bulk_threads(L) + 32 * cw; }
// Near quads per bulk thread (template parameter NEARQ): 0 = the bulk warps sum both halves everywhere.
__host__ __device__ inline int direct_nearq(int L, int r_hi) {
    const int njr = L / 64, off = direct_near_off(r_hi);
    const int nq = (off / 2 + 8 + njr - 1) / njr;
    if (off == 0 || L < 2 * off + 64 || nq > 4) return 0;
    return nq == 3 ? 4 : nq;
}
// dynamic smem (32-bit words): theta[L] | lut[2L] | lutb[2L] (q > 8 only) | sp[W] | sp0[W] | bq[W] | selb[L/4] | part[64] | Jz[96]
__host__ __device__ inline size_t direct_smem_bytes(int L, int q) {
    return (size_t)((q > 8 ? 5 : 3) * L + 3 * (L / 8) + L / 4 + 64 + 96) * 4;
}

__device__ __forceinline__ int dp4a_s32_u32(int a, uint32_t b, int c) {
    int d;
    asm("dp4a.s32.u32 %0, %1, %2, %3;" : "=r"(d) : "r"(a), "r"(b), "r"(c));
    return d;
}
// PRMT without the selector masking of __byte_perm (colours are < 8, so bit 3 of every selector nibble is 0;
// selector bits above 15 are ignored by the instruction)
__device__ __forceinline__ uint32_t prmt(uint32_t a, uint32_t b, uint32_t sel) {
    uint32_t d;
    asm("prmt.b32 %0, %1, %2, %3;" : "=r"(d) : "r"(a), "r"(b), "r"(sel));
    return d;
}

// Colour -> s' lookup of 4 sites at once: the 4 colour nibbles of `sel` select bytes of the site's table.  Colours
// 8..15 (Q16) live in a second 8-byte table: a selector nibble with bit 3 set makes PRMT return the replicated sign
// bit of the selected byte, i.e. 0 for table bytes 0..2, so each PRMT contributes only its own half and the two
// results are OR-ed (selx = sel ^ 0x8888).
template <bool Q16>
__device__ __forceinline__ uint32_t tab_lookup(const uint2& ta, const uint2& tb, uint32_t sel, uint32_t selx) {
    uint32_t v = prmt(ta.x, ta.y, sel);
    if (Q16) v |= prmt(tb.x, tb.y, selx);
    return v;
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
    uint2* lut;       // [L]  per-site colour -> s' byte table, colours 0..7
    uint2* lutb;      // [L]  colours 8..15 (q > 8 only)
    uint32_t* sp;     // [W]  live packed spins
    uint32_t* sp0;    // [W]  spins at the start of the running sweep
    uint32_t* bq;     // [W]  proposed colours
    uint8_t* selb;    // [L]  a0 | b << 4: colour at the start of the sweep and proposed colour
    uint32_t* part;   // [2][32] block sums S_i, double buffered
    int32_t* Jz;      // [96] Jz[n] = 0 for n < 32, Jq[n - 32] above
};

// Start of a sweep, all threads: proposals, thresholds and colour tables of all sites (A6, A7, A9) and the
// snapshot of the spins.
template <bool Q16>
__device__ __forceinline__ void direct_draw(const Dev& d, const DirectSmem& m, uint32_t sweep, int t, uint32_t c3,
                                            double scale) {
    const int W = d.W, q = d.q;
    // one work item = 4 sites (half a packed word): 2W items over all threads of the CTA
    for (int hw = threadIdx.x; hw < 2 * W; hw += blockDim.x) {
        const int w = hw >> 1, h4 = (hw & 1) << 2;
        const uint32_t word = m.sp[w];
        uint32_t bhalf = 0, s4 = 0;
#pragma unroll
        for (int n = 0; n < 4; ++n) {
            const int i = 8 * w + h4 + n;
            const Philox4 p = philox4x32_10((uint32_t)i, sweep, (uint32_t)t, c3, d.key0, d.key1);
            const uint32_t a = (word >> (4 * (h4 + n))) & 15u;
            const uint32_t k = __umulhi(p.w0, (uint32_t)(q - 1));
            const uint32_t b = k + (k >= a ? 1u : 0u);
            bhalf |= b << (4 * n);
            s4 |= (a | (b << 4)) << (8 * n);
            m.theta[i] = min(accept_threshold(uniform53(p.w1, p.w2), scale), 1 << 30);  // |dE| < 2^30: same decisions
            unsigned long long ta = 0x0101010101010101ull, tb = ta;   // byte k = s'(k), k = 0..7 | 8..15
            if (!Q16 || a < 8u) ta += 1ull << (8 * a); else tb += 1ull << (8 * (a - 8u));
            if (!Q16 || b < 8u) ta -= 1ull << (8 * b); else tb -= 1ull << (8 * (b - 8u));
            m.lut[i] = make_uint2((uint32_t)ta, (uint32_t)(ta >> 32));
            if (Q16) m.lutb[i] = make_uint2((uint32_t)tb, (uint32_t)(tb >> 32));
        }
        reinterpret_cast<uint16_t*>(m.bq)[hw] = (uint16_t)bhalf;   // low half of word w = sites 8w .. 8w+3
        reinterpret_cast<uint32_t*>(m.selb)[hw] = s4;
        if (h4 == 0) m.sp0[w] = word;
    }
}

// N_max of the configuration (Eq. 10): per-thread colour counts in registers, one warp reduction and one shared-memory
// atomic per colour and warp.  Called by all threads (cta_sync inside); every thread gets the result.
__device__ __forceinline__ int direct_nmax(const uint32_t* sp, int W, int q, int* s_cnt) {
    if (threadIdx.x < 16) s_cnt[threadIdx.x] = 0;
    cta_sync();
    int cnt[16];
#pragma unroll
    for (int k = 0; k < 16; ++k) cnt[k] = 0;
    for (int w = threadIdx.x; w < W; w += blockDim.x) {
        const uint32_t word = sp[w];
#pragma unroll
        for (int k = 0; k < 16; ++k)
            if (k < q) cnt[k] += __popc(match_nibbles(word, (uint32_t)k));
    }
#pragma unroll
    for (int k = 0; k < 16; ++k) {
        if (k < q) {
            const int c = __reduce_add_sync(0xffffffffu, cnt[k]);
            if ((threadIdx.x & 31) == 0 && c) atomicAdd(&s_cnt[k], c);
        }
    }
    cta_sync();
    int nmax = 0;
    for (int k = 0; k < q; ++k) nmax = max(nmax, s_cnt[k]);   // every thread: whoever needs it has it
    return nmax;
}

// Swap event inside a persistent launch (all CTAs of the ensemble co-resident: cooperative launch; n_rep <=
// DIRECT_MAX_PERSIST_REP).  Nothing is serialised in one CTA: every CTA publishes its energy (Epub, double buffered by
// event parity), arrives on the ensemble's counter gen[e] (zeroed by the host before the launch), waits until all
// n_rep arrivals of this event are in, fetches all energies and evaluates the whole event (Eq. 9; even pairs, then odd
// pairs) on its OWN copy of the slot -> storage permutation in shared memory: the decisions are a pure
// function of (energies, permutation, Philox(slot, sweep)), so all copies stay identical.  The CTA that holds storage 0
// also counts the attempts/acceptances.  Returns the slot the configuration with storage index st now occupies.
// Called by ALL threads of the CTA.
// Waits (acquire) until the arrival counter *cnt reaches target.  The wait is bounded by wall-clock time (%globaltimer,
// nanoseconds), not by a number of polls: a co-resident CTA may legitimately be late by a long time (time slicing with
// another process, a profiler replaying the kernel).  After DIRECT_BARRIER_TIMEOUT_NS, or as soon as another CTA has
// given up, *err is raised (pt_sync then returns PT_ECUDA; the state of the context is lost) and the wait returns.
constexpr unsigned long long DIRECT_BARRIER_TIMEOUT_NS = 30ull * 1000ull * 1000ull * 1000ull;
__device__ __forceinline__ void wait_arrivals(const unsigned* cnt, unsigned target, int* err) {
    unsigned g = 0u, polls = 0u;
    unsigned long long t0 = 0ull;
    while (true) {
        asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(g) : "l"(cnt) : "memory");
        if (g >= target) return;
        if ((++polls & 1023u) == 0u) {
            unsigned long long now;
            asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(now));
            if (t0 == 0ull) t0 = now;
            if (now - t0 > DIRECT_BARRIER_TIMEOUT_NS || *(volatile int*)err != 0) {
                *(volatile int*)err = 1;
                return;
            }
        }
    }
}

struct PersistSmem {
    int* perm;          // [n_rep] slot -> storage
    long long* Eall;    // [n_rep] energies by storage index
    int* slot;          // result
};
__device__ __forceinline__ int direct_swap_in_kernel(const Dev& d, const PersistSmem& ps, int e, uint32_t sweep, int st,
                                                     const long long* s_E, int event) {
    const int n_rep = d.n_rep;
    long long* Epub = d.Epub + ((size_t)(event & 1) * d.n_ens + e) * n_rep;
    if (threadIdx.x == 0) {
        __stcg(Epub + st, *s_E);
        // release: the energy is visible to whoever observes the arrival (cheaper than a full __threadfence)
        asm volatile("red.release.gpu.global.add.u32 [%0], 1;" ::"l"(d.gen + e) : "memory");
        wait_arrivals(d.gen + e, (unsigned)n_rep * (unsigned)(event + 1), d.err);
    }
    cta_sync();
    for (int t2 = threadIdx.x; t2 < n_rep; t2 += blockDim.x) ps.Eall[t2] = __ldcg(Epub + t2);
    cta_sync();
    const uint32_t c3 = ((uint32_t)(d.ens_base + e) << 4) | TAG_SWAP;
    pt_obs* obs = d.obs + (size_t)e * n_rep;
    for (int stage = 0; stage < 2; ++stage) {
        for (int t2 = stage + 2 * (int)threadIdx.x; t2 + 1 < n_rep; t2 += 2 * (int)blockDim.x) {
            const int sa = ps.perm[t2], sb = ps.perm[t2 + 1];
            const double dd = __dmul_rn(d.beta[t2] - d.beta[t2 + 1], ldexp((double)(ps.Eall[sa] - ps.Eall[sb]), -24));
            const Philox4 p = philox4x32_10((uint32_t)t2, sweep, 0u, c3, d.key0, d.key1);
            const bool acc = dd >= 0.0 || uniform53(p.w1, p.w2) < exp(dd);
            if (acc) { ps.perm[t2] = sb; ps.perm[t2 + 1] = sa; }
            if (st == 0) {
                atomicAdd((unsigned long long*)&obs[t2].swap_attempts, 1ull);
                if (acc) atomicAdd((unsigned long long*)&obs[t2].swap_accepts, 1ull);
            }
        }
        cta_sync();
    }
    for (int t2 = threadIdx.x; t2 < n_rep; t2 += blockDim.x)
        if (ps.perm[t2] == st) *ps.slot = t2;
    cta_sync();
    return *ps.slot;
}

#ifdef PT_TIMING
#define PT_T0(v) const long long v = clock64()
#define PT_ACC(slot, v) tacc[slot] += clock64() - (v)
#else
#define PT_T0(v)
#define PT_ACC(slot, v)
#endif

// sum over the 4 bits b..b+3 of m of (bit ? c : 0), added to acc: 4 LOP3 (bit test -> predicate), 4 SEL, 2 IADD3,
// all on the ALU pipe (the compiler's own choice for this pattern is shift pairs on the FMA or uniform pipes)
__device__ __forceinline__ int masked_add4(int acc, unsigned m, int b, int4 c) {
    asm("{\n\t.reg .pred p0, p1, p2, p3;\n\t.reg .b32 t0, t1, t2, t3;\n\t"
        "and.b32 t0, %5, %6;\n\tsetp.ne.u32 p0, t0, 0;\n\t"
        "and.b32 t1, %5, %7;\n\tsetp.ne.u32 p1, t1, 0;\n\t"
        "and.b32 t2, %5, %8;\n\tsetp.ne.u32 p2, t2, 0;\n\t"
        "and.b32 t3, %5, %9;\n\tsetp.ne.u32 p3, t3, 0;\n\t"
        "selp.b32 t0, %1, 0, p0;\n\tselp.b32 t1, %2, 0, p1;\n\tselp.b32 t2, %3, 0, p2;\n\tselp.b32 t3, %4, 0, p3;\n\t"
        "add.s32 t0, t0, t1;\n\tadd.s32 t2, t2, t3;\n\tadd.s32 t0, t0, t2;\n\tadd.s32 %0, %0, t0;\n\t}"
        : "+r"(acc)
        : "r"(c.x), "r"(c.y), "r"(c.z), "r"(c.w), "r"(m), "r"(1u << b), "r"(2u << b), "r"(4u << b), "r"(8u << b));
    return acc;
}

// ---- mbarrier (shared-memory transaction barrier) helpers: producer/consumer hand-off between the warps ----
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
// release: the arriving thread's earlier shared-memory writes are visible to whoever sees the phase complete
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
    asm volatile("{\n\t.reg .b64 st;\n\tmbarrier.arrive.shared::cta.b64 st, [%0];\n\t}" ::"r"(smem_u32(bar)) : "memory");
}
// blocks until the phase with the given parity has completed (acquire)
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "MBAR_WAIT:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
        "@p bra MBAR_DONE;\n\t"
        "bra MBAR_WAIT;\n\t"
        "MBAR_DONE:\n\t}" ::"r"(smem_u32(bar)), "r"(parity)
        : "memory");
}

// FAR (template parameter; L = 4096, q <= 8, one near quad per thread, and d.far: checked by the host).  Beyond a
// distance of about 1000 sites the couplings a bulk thread holds differ from their minimum Jmin by less than 256.
// With Jq = Jmin + res,
//   sum_j Jq[i-j] s'_i(c_j) = sum_j res[i-j] s'_i(c_j) + Jmin (32 + n_a - n_b),
// n_c = sites of colour c among the 32 of the range: the first sum takes ONE IDP.4A per four pair terms (8-bit
// residuals) instead of two IDP.2A, the second is a look-up in the colour counts of the range's block (one PRMT +
// one IDP.2A per site).  So that every bulk warp gains the same, every thread takes half a near range and half a far
// range: thread (g, jr) sums the 32 sites j of block kb + jr (jr < 32) resp. kb + 64 + jr (the near half: distances
// below 1024, IDP.2A on 16-bit halves as before) and the 32 sites of block kb + 32 + jr (the far half).  The counts
// of a block (s_cnt8: 8 bytes, colours 0..7) are recounted by a bulk warp when the block has been decided; a far
// range is at least 31 blocks away from the blocks in flight.
__device__ __forceinline__ uint32_t dp2a_lo_s32_u32(uint32_t a, uint32_t b, uint32_t c) {
    uint32_t d;
    asm("dp2a.lo.s32.u32 %0, %1, %2, %3;" : "=r"(d) : "r"(a), "r"(b), "r"(c));
    return d;
}
__device__ __forceinline__ uint32_t dp4a_u32_u32(uint32_t a, uint32_t b, uint32_t c) {
    uint32_t d;
    asm("dp4a.u32.u32 %0, %1, %2, %3;" : "=r"(d) : "r"(a), "r"(b), "r"(c));
    return d;
}
// one warp: colour counts of block blk (4 words) -> cnt8[blk]
__device__ __forceinline__ void recount_block(const uint32_t* sp, uint2* cnt8, int blk, int lane) {
    const uint32_t x = sp[4 * blk + (lane >> 3)];
    int v = __popc(match_nibbles(x, (uint32_t)(lane & 7)));
    v += __shfl_xor_sync(0xffffffffu, v, 8);
    v += __shfl_xor_sync(0xffffffffu, v, 16);
    if (lane < 8) reinterpret_cast<uint8_t*>(cnt8 + blk)[lane] = (uint8_t)v;
}

// NEARQ = 0: the bulk warps sum both 16-bit halves of every coupling.  NEARQ = 1, 2, 4: they sum the low halves
// only, plus the high halves of NEARQ of the off/2 + 8 quads of sites within distance off - 1 of the block (requires
// r_hi < off = direct_near_off(r_hi) and NEARQ * L/64 >= off/2 + 8).  NJR64: L == 4096 (64 j-ranges as a compile-time
// constant).
// MINB: minimum CTAs per SM the register allocation must allow (1: up to 168 registers, for large L; 2: 80 registers,
// so that several hundred small replicas can be co-resident for persistent launches); 3 stands for the L > 4096
// build: one CTA of up to DIRECT_BIG_THREADS threads per SM, 80 registers.
// MINB = 4 stands for the L <= 2048 build: CTAs of at most DIRECT_MID_THREADS threads, two per SM, 128 registers.
// WIDE: the near window is direct_near_off(r_hi) = 160 .. 352 sites (a run-time value); else 96 (compile-time: the
// schedule of the headline instantiation is sensitive to every instruction).
// CW: chain warps (4: one per SM sub-partition, 8 correction rows each; 2: 16 rows each -- 25 % fewer chain
// instructions per block but longer fixed-point rounds).  Measured (profiles/r2_f_two_ctas_per_sm.md): two chain
// warps are slower wherever tried -- configs[3] 0.1667 against 0.1419 ms per sweep, configs[4] 0.71 against 0.54 with
// two 192-thread CTAs per SM at 168 registers, L = 2048 x 296..1200 replicas +0.5..+7 % -- the chain's serial latency,
// not its instruction count, is what a block waits for.  Kept as an opt-in experiment of the headline instantiation
// (PT_CW=2, bit-identical results).
template <int NEARQ, bool NJR64, bool Q16, int MINB, bool FAR = false, bool WIDE = false, int CW = DIRECT_CHAIN_WARPS>
__global__ void __launch_bounds__(MINB == 3 ? DIRECT_BIG_THREADS
                                  : MINB == 4 ? DIRECT_MID_THREADS - 32 * (DIRECT_CHAIN_WARPS - CW)
                                              : DIRECT_MAX_THREADS - 32 * (DIRECT_CHAIN_WARPS - CW),
                                  MINB == 3 ? 1 : MINB == 4 ? 2 : MINB)
sweep_direct_kernel(Dev d, long long sweep0, int n_sweeps, int swap_mode, int swap_every, int r_hi) {
    // swap_mode 0: no swap event; 1: one event at the end of the launch (last-arriving CTA, nobody waits);
    // 2: persistent launch, an event inside the kernel after every sweep whose index is a multiple of swap_every;
    // 3: slot-sharded context (one ensemble): CTA b sweeps the configuration with storage index rep_base + b at
    //    whatever slot it occupies now; no swap event (the caller exchanges energies and calls pt_swap_external).
    constexpr bool FULL_HI = NEARQ == 0;
    constexpr int NQ = NEARQ ? NEARQ : 1;
    extern __shared__ uint32_t smem_d[];
    const int L = d.L, W = d.W, q = d.q;
    const int NT = blockDim.x, NTB = NT - 32 * CW;
    const int NB = L >> 5;
    DirectSmem m;
    m.theta = (int32_t*)smem_d;
    m.lut = (uint2*)(m.theta + L);
    m.lutb = m.lut + L;
    m.sp = (uint32_t*)(m.lut + (Q16 ? 2 * L : L));
    m.sp0 = m.sp + W;
    m.bq = m.sp0 + W;
    m.selb = (uint8_t*)(m.bq + W);
    m.part = (uint32_t*)(m.selb + L);
    m.Jz = (int32_t*)(m.part + 64);
    __shared__ int s_cnt[16];
    __shared__ long long s_E;   // running energy of this configuration (owner: lane 0 of chain warp 0)
    __shared__ int s_slot;
    __shared__ ObsAcc s_oa;
    __shared__ int s_perm[DIRECT_MAX_PERSIST_REP];
    __shared__ long long s_Eall[DIRECT_MAX_PERSIST_REP];
    __shared__ double s_scale[DIRECT_MAX_PERSIST_REP];
    PersistSmem ps;
    ps.perm = s_perm; ps.Eall = s_Eall; ps.slot = &s_slot;
    int event = 0;   // swap events so far in this (persistent) launch
    // full[s]: the block sums of buffer s are complete (one arrival per bulk warp);
    // done[s]: the chain warps have decided the block of buffer s and written its spins (one arrival).
    __shared__ __align__(8) uint64_t s_full[2], s_done[2];
    __shared__ __align__(16) int s_xch[2][32][4];   // partial sums exchanged between the chain warps
    __shared__ uint2 s_cnt8[128];                   // FAR: colour counts of the 32-site blocks

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int e = swap_mode == 3 ? 0 : blockIdx.x / d.n_rep;
    int t = blockIdx.x % d.n_rep;   // slot (temperature) of this CTA's configuration; moves in swap_mode 2
    // state that the previous launch wrote (perm, spins, E) and, for persistent launches, the ensemble's tables
    size_t x = 0;
    int st = 0;
    uint32_t* g_sp = nullptr;
#define PT_LOAD_STATE()                                             \
    do {                                                                     \
        st = swap_mode == 3 ? d.rep_base + (int)blockIdx.x : d.perm[blockIdx.x];  \
        if (swap_mode == 3)                                                  \
            for (int t2 = tid; t2 < d.n_rep; t2 += NT)                       \
                if (d.perm[t2] == st) s_slot = t2;                           \
        x = (size_t)e * d.n_rep + st;                                        \
        g_sp = d.spins + x * W;                                              \
        for (int w = tid; w < W; w += NT) m.sp[w] = g_sp[w];                 \
        if (swap_mode == 2)                                                  \
            for (int t2 = tid; t2 < d.n_rep; t2 += NT) {                     \
                s_perm[t2] = d.perm[(size_t)e * d.n_rep + t2];               \
                s_scale[t2] = d.thr_scale[t2];                               \
            }                                                                \
    } while (0)
#ifdef PT_TIMING
    long long tacc[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    PT_T0(t_kernel);
    unsigned long long gt_start;   // wall clock (ns) at the first instruction: launch gaps = start(n+1) - end(n)
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(gt_start));
#endif

    for (int n = tid; n < 96; n += NT) m.Jz[n] = n < 32 ? 0 : d.Jq[n - 32];
    if (tid < 64) m.part[tid] = 0u;
    double scale = d.thr_scale[t];
    const uint32_t c3 = ((uint32_t)(d.ens_base + e) << 4) | TAG_SWEEP;

    if (tid < NTB) {
        // =========================== BULK warps ===========================
        // thread -> (site group g, j-range jr); group g = the 8 sites 16(g>>1) + (g&1) + {0,2,..,14}
        const int g = tid & 3, jr = tid >> 2;
        const int par = g & 1, gbase = 16 * (g >> 1) + par;
        const int NJR = NJR64 ? 64 : L / 64;
        const bool active = jr < NJR;
        // couplings of this thread: pair tt holds Jq[r], Jq[r-1] with r = R0 - 2 tt  (mod L)
        constexpr int NPL = FAR ? 45 : DIRECT_NPAIR;   // FAR: 23 pairs of the near half, 22 fours of the far half
        uint32_t PL[NPL];
        uint32_t PH[FULL_HI ? DIRECT_NPAIR : 1];
        uint32_t jpm = 0u, jmin32 = 0u;   // FAR: Jmin | -Jmin << 16 and 32 Jmin of the far half
        // FAR: first site of the near half and of the far half, relative to the block start
        const int jn = jr < 32 ? 32 * jr : L - 1024 + 32 * (jr - 32), jf = 1024 + 32 * jr;
        if (FAR) {
            {   // near half: pair tt holds the low halves of Jq[r], Jq[r-1], r = R0 - 2 tt (mod L)
                const int H = L / 2;
                const uint32_t* lo = d.Jpair + (size_t)(2 * par) * H;
                int r = ((gbase + 14 - jn) % L + L) % L;
#pragma unroll
                for (int tt = 0; tt < 23; ++tt) {
                    PL[tt] = __ldg(lo + ((r - par) >> 1));
                    r -= 2;
                    r += r < 0 ? L : 0;
                }
            }
            {   // far half: four tt holds Jq[r] - Jmin, .., Jq[r-3] - Jmin, r = R0 - 2 tt (mod L), one byte each
                const int R0 = ((gbase + 14 - jf) % L + L) % L;
                int jmin = 0x7fffffff;
                for (int n = 0; n < 46; ++n) {
                    int r = R0 - n;
                    r += r < 0 ? L : 0;
                    jmin = min(jmin, __ldg(d.Jq + r));
                }
                int r = R0;
#pragma unroll
                for (int tt = 0; tt < 22; ++tt) {
                    uint32_t qd = 0u;
#pragma unroll
                    for (int c = 0; c < 4; ++c) {
                        int rc = r - c;
                        rc += rc < 0 ? L : 0;
                        qd |= (uint32_t)(__ldg(d.Jq + rc) - jmin) << (8 * c);
                    }
                    PL[23 + tt] = qd;
                    r -= 2;
                    r += r < 0 ? L : 0;
                }
                jpm = ((uint32_t)jmin & 0xffffu) | ((uint32_t)(-jmin) << 16);
                jmin32 = 32u * (uint32_t)jmin;
            }
            PH[0] = 0u;
        } else {
            const int H = L / 2;
            const int R0 = ((gbase + 14 - 64 * jr) % L + L) % L;
            const uint32_t* lo = d.Jpair + (size_t)(2 * par) * H;
            const uint32_t* hi = lo + H;
            int r = R0;   // r = R0 - 2 tt (mod L) keeps the parity of `par`: no division or modulo per load
#pragma unroll
            for (int tt = 0; tt < DIRECT_NPAIR; ++tt) {
                const int mm = (r - par) >> 1;
                PL[tt] = active ? __ldg(lo + mm) : 0u;
                if (FULL_HI) PH[tt] = active ? __ldg(hi + mm) : 0u;
                r -= 2;
                r += r < 0 ? L : 0;
            }
            if (!FULL_HI) PH[0] = 0u;
        }
        // NEAR: high halves of quad n = jr + NJR*iq (sites i0 - NOFF + 4n + {0..3}) for this thread's 8 sites:
        // NP[iq][mm][0] = hi(|r|) | hi(|r-1|) << 16, [1] = hi(|r-2|) | hi(|r-3|) << 16, r = gbase + 2mm + NOFF - 4n,
        // hi(x) = Jq[x] >> 16 for 1 <= x <= r_hi, else 0.  NOFF = 96 .. 352 sites (direct_near_off), NQD quads.
        const int NOFF = (NEARQ && WIDE) ? direct_near_off(r_hi) : 96, NQD = NOFF / 2 + 8;
        uint32_t NP[NQ][DIRECT_SITES][2];
        if (NEARQ) {
#pragma unroll
            for (int iq = 0; iq < NQ; ++iq) {
                const int n = jr + NJR * iq;
#pragma unroll
                for (int mm = 0; mm < DIRECT_SITES; ++mm) {
                    uint32_t hv[4];
#pragma unroll
                    for (int c = 0; c < 4; ++c) {
                        int r = gbase + 2 * mm + NOFF - 4 * n - c;
                        r = r < 0 ? -r : r;
                        hv[c] = (active && n < NQD && r >= 1 && r <= r_hi) ? ((uint32_t)__ldg(d.Jq + r) >> 16)
                                                                                        : 0u;
                    }
                    NP[iq][mm][0] = hv[0] | (hv[1] << 16);
                    NP[iq][mm][1] = hv[2] | (hv[3] << 16);
                }
            }
        }
        PT_LOAD_STATE();
        if (tid == 0) {
            mbar_init(&s_full[0], NTB >> 5); mbar_init(&s_full[1], NTB >> 5);
            mbar_init(&s_done[0], 1); mbar_init(&s_done[1], 1);
        }
        cta_sync();
        if (swap_mode == 3) { t = s_slot; scale = d.thr_scale[t]; }
        if (FAR)   // colour counts of all blocks (read after the barrier that follows the first DRAW)
            for (int blk = warp; blk < NB; blk += NTB >> 5) recount_block(m.sp, s_cnt8, blk, lane);

        for (int s = 0; s < n_sweeps; ++s) {
            PT_T0(t_draw);
            direct_draw<Q16>(d, m, (uint32_t)(sweep0 + s + 1), t, c3, scale);
            cta_sync();
            PT_ACC(0, t_draw);
            // the four barriers are initialised once per launch; every sweep completes NB/2 phases of each
            const int phase0 = s * (NB >> 1);
            PT_T0(t_loop);
            // per-thread cursors, advanced by one block (32 sites = 4 words) per block
            const uint2* lutp = m.lut + gbase;   // (table of colours 8..15: L entries further)
            int wj = FAR ? jn >> 3 : 8 * jr;                    // first word of this thread's j-range (FAR: of its near half)
            int wjf = jf >> 3;                                  // FAR: first word of the far half
            // the second half of the last range is block kb-1, which is being decided: sweep-start copy
            // (FAR: the near half of jr = 63 IS block kb-1)
            const uint32_t* sp2 = (jr == NJR - 1) ? m.sp0 : m.sp;
            int wn[NQ];                                         // NEAR: word of quad n = jr + NJR*iq
#pragma unroll
            for (int iq = 0; iq < NQ; ++iq) {
                wn[iq] = ((jr + NJR * iq) >> 1) - (NOFF >> 3);
                wn[iq] += wn[iq] < 0 ? W : 0;
            }
            for (int kb = 0; kb < NB; ++kb) {
                // block kb is summed against: blocks < kb-1 final (the chain warp is done with block kb-2, which
                // also frees buffer kb&1), block kb-1 as at the start of the sweep, blocks >= kb untouched
#ifdef PT_TIMING
                if (kb >= 2) {   // slot 5: try_waits that found the phase incomplete; slot 6 (below): clocks of the wait
                    PT_T0(t_w);
                    uint32_t ok = 0u;
                    do {
                        asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
                                     "selp.u32 %0, 1, 0, p;\n\t}"
                                     : "=r"(ok) : "r"(smem_u32(&s_done[kb & 1])), "r"((uint32_t)(phase0 + (kb >> 1) - 1) & 1u) : "memory");
                        tacc[5] += ok ? 0 : 1;
                    } while (!ok);
                    PT_ACC(7, t_w);
                }
#else
                if (kb >= 2) mbar_wait(&s_done[kb & 1], (uint32_t)(phase0 + (kb >> 1) - 1) & 1u);
#endif
                PT_T0(t_b);
                // FAR: block kb-2 is final: its colour counts (a far range reads them 30 blocks later at the earliest)
                int rcv = 0;
                if (FAR && kb >= 2 && warp == (kb & 7))
                    rcv = __popc(match_nibbles(m.sp[4 * (kb - 2) + (lane >> 3)], (uint32_t)(lane & 7)));
                uint32_t val[DIRECT_SITES] = {0u, 0u, 0u, 0u, 0u, 0u, 0u, 0u};
                if (active) {
                    int wj2 = wj + 4;
                    wj2 -= wj2 >= W ? W : 0;
                    const uint4 wa = *reinterpret_cast<const uint4*>((FAR ? sp2 : m.sp) + wj);
                    const uint4 wb = *reinterpret_cast<const uint4*>(FAR ? m.sp + wjf : sp2 + wj2);
                    const uint32_t words[8] = {wa.x, wa.y, wa.z, wa.w, wb.x, wb.y, wb.z, wb.w};   // FAR: near half | far half
                    uint2 lt[DIRECT_SITES], ltb[DIRECT_SITES];
#pragma unroll
                    for (int mm = 0; mm < DIRECT_SITES; ++mm) {
                        lt[mm] = lutp[2 * mm];
                        ltb[mm] = Q16 ? lutp[L + 2 * mm] : make_uint2(0u, 0u);
                    }
                    uint32_t nword[NQ];
#pragma unroll
                    for (int iq = 0; iq < NQ; ++iq) {   // the 8 quads before quad NOFF/4 are block kb-1: sweep-start copy
                        const int n = jr + NJR * iq;
                        nword[iq] = NEARQ ? ((n >= (NOFF >> 2) - 8 && n < (NOFF >> 2)) ? m.sp0 : m.sp)[wn[iq]] : 0u;
                    }
                    // two accumulators per site (even / odd pair of j) keep the IDP.2A chains short
                    uint32_t alo[DIRECT_SITES], alo2[DIRECT_SITES], ahi[DIRECT_SITES];
#pragma unroll
                    for (int mm = 0; mm < DIRECT_SITES; ++mm) { alo[mm] = 0u; alo2[mm] = 0u; ahi[mm] = 0u; }
                    if (FAR) {
                        // far half, Jmin (32 + n_a - n_b) from the colour counts of its block
                        int B = kb + 32 + jr;
                        B -= B >= NB ? NB : 0;
                        const uint2 cn = s_cnt8[B];
                        const uint4 sb = *reinterpret_cast<const uint4*>(m.selb + (kb << 5) + 16 * (g >> 1));
                        const uint32_t sbw[4] = {sb.x >> (8 * par), sb.y >> (8 * par), sb.z >> (8 * par), sb.w >> (8 * par)};
#pragma unroll
                        for (int mm = 0; mm < DIRECT_SITES; ++mm) {
                            // byte of site gbase + 2 mm: a | b << 4 -> PRMT bytes 0, 1 = counts of a, b
                            const uint32_t selc = (mm & 1) ? (sbw[mm >> 1] >> 16) : sbw[mm >> 1];
                            alo[mm] = dp2a_lo_s32_u32(jpm, prmt(cn.x, cn.y, selc), jmin32);
                        }
                        // near half: as below, 8 steps of four sites
#pragma unroll
                        for (int u = 0; u < 8; ++u) {
                            const uint32_t sel = (u & 1) ? (words[u >> 1] >> 16) : words[u >> 1];
#pragma unroll
                            for (int mm = 0; mm < DIRECT_SITES; ++mm) {
                                const uint32_t S = prmt(lt[mm].x, lt[mm].y, sel);
                                const int tt = 7 - mm + 2 * u;
                                alo[mm] = __dp2a_lo(PL[tt], S, alo[mm]);
                                alo2[mm] = __dp2a_hi(PL[tt + 1], S, alo2[mm]);
                            }
                        }
                        // far half, residual sums: one IDP.4A per four pair terms
#pragma unroll
                        for (int u = 0; u < 8; ++u) {
                            const uint32_t sel = (u & 1) ? (words[4 + (u >> 1)] >> 16) : words[4 + (u >> 1)];
#pragma unroll
                            for (int mm = 0; mm < DIRECT_SITES; ++mm) {
                                uint32_t& acc = (u & 1) ? alo2[mm] : alo[mm];
                                acc = dp4a_u32_u32(PL[23 + 7 - mm + 2 * u], prmt(lt[mm].x, lt[mm].y, sel), acc);
                            }
                        }
                    } else {
#pragma unroll
                    for (int u = 0; u < 16; ++u) {
                        const uint32_t sel = (u & 1) ? (words[u >> 1] >> 16) : words[u >> 1];
                        const uint32_t selx = sel ^ 0x8888u;
#pragma unroll
                        for (int mm = 0; mm < DIRECT_SITES; ++mm) {
                            const uint32_t S = tab_lookup<Q16>(lt[mm], ltb[mm], sel, selx);
                            const int tt = 7 - mm + 2 * u;
                            alo[mm] = __dp2a_lo(PL[tt], S, alo[mm]);
                            alo2[mm] = __dp2a_hi(PL[tt + 1], S, alo2[mm]);
                            if (FULL_HI) {
                                ahi[mm] = __dp2a_lo(PH[FULL_HI ? tt : 0], S, ahi[mm]);
                                ahi[mm] = __dp2a_hi(PH[FULL_HI ? tt + 1 : 0], S, ahi[mm]);
                            }
                        }
                    }
                    }
                    if (NEARQ) {
#pragma unroll
                        for (int iq = 0; iq < NQ; ++iq) {
                            const int n = jr + NJR * iq;
                            const uint32_t sel = (n & 1) ? (nword[iq] >> 16) : nword[iq];
#pragma unroll
                            for (int mm = 0; mm < DIRECT_SITES; ++mm) {
                                const uint32_t S = tab_lookup<Q16>(lt[mm], ltb[mm], sel, sel ^ 0x8888u);
                                ahi[mm] = __dp2a_lo(NP[iq][mm][0], S, ahi[mm]);
                                ahi[mm] = __dp2a_hi(NP[iq][mm][1], S, ahi[mm]);
                            }
                        }
                    }
#pragma unroll
                    for (int mm = 0; mm < DIRECT_SITES; ++mm) val[mm] = alo[mm] + alo2[mm] + (ahi[mm] << 16);
                    // advance the cursors
                    lutp += 32;
                    wj += 4;
                    wj -= wj >= W ? W : 0;
                    wjf += 4;
                    wjf -= wjf >= W ? W : 0;
#pragma unroll
                    for (int iq = 0; iq < NQ; ++iq) {
                        wn[iq] += 4;
                        wn[iq] -= wn[iq] >= W ? W : 0;
                    }
                }
                // block sums: transpose-reduce over the 8 lanes of a warp that hold the same site group (lane bits
                // 2..4 = j-range): 4 + 2 + 1 shuffles leave one site per lane, m = lane bits (2,3,4), then one
                // shared-memory atomic per lane (32 different sites per warp)
                {
                    uint32_t v4[4], v2[2];
                    const bool u4 = lane & 16, u3 = lane & 8, u2 = lane & 4;
#pragma unroll
                    for (int i = 0; i < 4; ++i)
                        v4[i] = (u4 ? val[i + 4] : val[i]) + __shfl_xor_sync(0xffffffffu, u4 ? val[i] : val[i + 4], 16);
#pragma unroll
                    for (int i = 0; i < 2; ++i)
                        v2[i] = (u3 ? v4[i + 2] : v4[i]) + __shfl_xor_sync(0xffffffffu, u3 ? v4[i] : v4[i + 2], 8);
                    const uint32_t v1 = (u2 ? v2[1] : v2[0]) + __shfl_xor_sync(0xffffffffu, u2 ? v2[0] : v2[1], 4);
                    const int msite = (u2 ? 1 : 0) + (u3 ? 2 : 0) + (u4 ? 4 : 0);
                    atomicAdd(&m.part[(kb & 1) * 32 + gbase + 2 * msite], v1);
                }
                __syncwarp();
                if (lane == 0) mbar_arrive(&s_full[kb & 1]);
                if (FAR && kb >= 2 && warp == (kb & 7)) {   // behind the arrival: nobody waits for this
                    rcv += __shfl_xor_sync(0xffffffffu, rcv, 8);
                    rcv += __shfl_xor_sync(0xffffffffu, rcv, 16);
                    if (lane < 8) reinterpret_cast<uint8_t*>(s_cnt8 + kb - 2)[lane] = (uint8_t)rcv;
                }
                PT_ACC(1, t_b);
            }
            PT_ACC(2, t_loop);
            PT_T0(t_end);
            cta_sync();  // the chain warp has decided the last block and published its sums
            if (FAR && warp < 2) recount_block(m.sp, s_cnt8, NB - 2 + warp, lane);
            PT_ACC(6, t_end);
            PT_T0(t_nm);
            // a8 (the chain warps' owner thread samples the observables; every thread helps counting colours)
            direct_nmax(m.sp, W, q, s_cnt);
            cta_sync();
            PT_ACC(6, t_nm);   // (slot 6: the closing barrier and the colour count; slot 7 is the done wait)
            if (swap_mode == 2 && (sweep0 + s + 1) % swap_every == 0) {
                t = direct_swap_in_kernel(d, ps, e, (uint32_t)(sweep0 + s + 1), st, &s_E, event++);
                scale = s_scale[t];
            }
            PT_ACC(3, t_end);
        }
#ifdef PT_TIMING
        if (lane == 0 && d.dbg) {
            tacc[4] = clock64() - t_kernel;
            for (int n = 0; n < 8; ++n) d.dbg[((size_t)blockIdx.x * 32 + warp) * 8 + n] += tacc[n];
        }
#endif
    } else {
        // =========================== CHAIN warps ===========================
        // Four warps, one per SM sub-partition (a warp gets about a fifth of its scheduler's issue slots next to
        // four bulk warps, so the work of a block is spread over all four schedulers).  Every warp keeps the
        // slack y_l of all 32 sites (lane = site); warp cw owns the correction rows f = 8cw..8cw+7 and adds
        // their part of every masked sum; the parts are exchanged through shared memory (named barrier 1).
        const int cw = warp - (NTB >> 5);
        const uint32_t rowsum = d.rowsum;   // sum_r Jq[r], known to the host since pt_create
        // CORR: this warp's correction rows for lane = site l.  If site f of the previous block (rows f = 8cw+j)
        // or of the own block (rows 32 + 8cw + j) accepts a_f -> b_f, dE_l changes by
        //   Jq[dist] (s'_l(b_f) - s'_l(a_f)),   dist = l + 32 - f  resp.  l - f  (nothing for dist <= 0).
        constexpr int ROWS = 32 / CW, RG = ROWS / 4;   // correction rows per chain warp, in groups of four
        int Jp[ROWS], Jo[ROWS];
#pragma unroll
        for (int j = 0; j < ROWS; ++j) {
            const int dp = lane + 32 - (ROWS * cw + j), dn = lane - (ROWS * cw + j);
            Jp[j] = __ldg(d.Jq + dp);               // 1 <= dp <= 63 < L
            Jo[j] = dn > 0 ? __ldg(d.Jq + dn) : 0;
        }
        PT_LOAD_STATE();
        // Owner of the configuration's running energy and of the slot's accumulators (a8): lane 0 of chain warp 0.
        // They live in shared memory, so nothing of this costs registers in the bulk path.
        const bool owner = cw == 0 && lane == 0;
        ObsAcc& oa = s_oa;
        if (owner) { oa = ObsAcc(); s_E = d.E[x]; }
        cta_sync();
        if (swap_mode == 3) { t = s_slot; scale = d.thr_scale[t]; }
        // A per-lane zero the compiler cannot see through: xor-ed into the accept masks it keeps the bit tests
        // on the ALU pipe (LOP3 -> predicate, SEL) instead of shift pairs on the FMA or uniform pipes.
        const unsigned lz = (unsigned)m.Jz[lane];
        int xb = 0;   // exchange buffer in use

        for (int s = 0; s < n_sweeps; ++s) {
            direct_draw<Q16>(d, m, (uint32_t)(sweep0 + s + 1), t, c3, scale);
            cta_sync();
            const int phase0 = s * (NB >> 1);
            long long dE_acc = 0;
            int n_acc = 0;
            uint32_t mp = 0u;   // accept mask of the previous block
            for (int k = 0; k < NB; ++k) {
                const int i0 = k << 5;
                // independent of the bulk: threshold, the words of the block for the final update, and the
                // correction rows (from the colours at the start of the sweep and the proposals: selb)
                const int th = m.theta[i0 + lane];
                const int wsp = (i0 >> 3) + (lane & 3);
                const uint32_t w_old = m.sp[wsp], w_new = m.bq[wsp];
                const uint2 tab = m.lut[i0 + lane];
                const uint2 tabb = Q16 ? m.lutb[i0 + lane] : make_uint2(0u, 0u);
                int ipv = i0 - 32 + ROWS * cw;
                ipv += ipv < 0 ? L : 0;
                uint32_t sfp[RG], sfo[RG];                                                   // a | b << 4 of ROWS sites
                if (CW == 4) {
                    const uint2 vp = *reinterpret_cast<const uint2*>(m.selb + ipv);
                    const uint2 vo = *reinterpret_cast<const uint2*>(m.selb + i0 + ROWS * cw);
                    sfp[0] = vp.x; sfp[1] = vp.y; sfo[0] = vo.x; sfo[1] = vo.y;
                } else {
                    const uint4 vp = *reinterpret_cast<const uint4*>(m.selb + ipv);
                    const uint4 vo = *reinterpret_cast<const uint4*>(m.selb + i0 + ROWS * cw);
                    sfp[0] = vp.x; sfp[1] = vp.y; sfp[RG - 2] = vp.z; sfp[RG - 1] = vp.w;
                    sfo[0] = vo.x; sfo[1] = vo.y; sfo[RG - 2] = vo.z; sfo[RG - 1] = vo.w;
                }
                int cp[ROWS], co[ROWS];
#pragma unroll
                for (int j = 0; j < ROWS; ++j) {
                    const uint32_t wp = sfp[j >> 2], wo = sfo[j >> 2];
                    // selector byte j: nibble 0 = a_f, nibble 1 = b_f (the two higher nibbles pick bytes that the
                    // dot product weights with 0); byte 0 of the result = s'_l(a_f), byte 1 = s'_l(b_f)
                    const uint32_t sp_ = wp >> (8 * (j & 3)), so_ = wo >> (8 * (j & 3));
                    cp[j] = Jp[j] * dp4a_s32_u32(0x000001ff, tab_lookup<Q16>(tab, tabb, sp_, sp_ ^ 0x8888u), 0);
                    co[j] = Jo[j] * dp4a_s32_u32(0x000001ff, tab_lookup<Q16>(tab, tabb, so_, so_ ^ 0x8888u), 0);
                }
                int4 cpv[RG], cov[RG];
#pragma unroll
                for (int gq = 0; gq < RG; ++gq) {
                    cpv[gq] = make_int4(cp[4 * gq], cp[4 * gq + 1], cp[4 * gq + 2], cp[4 * gq + 3]);
                    cov[gq] = make_int4(co[4 * gq], co[4 * gq + 1], co[4 * gq + 2], co[4 * gq + 3]);
                }
                // changes accepted in block k-1, which the bulk sum saw as it was before: this warp's rows, known
                // before the wait; they ride along with the first round below (one exchange less per block)
                int pc = 0;
                if (mp) {
                    const unsigned mv = (mp >> (ROWS * cw)) ^ lz;
#pragma unroll
                    for (int gq = 0; gq < RG; ++gq) pc = masked_add4(pc, mv, 4 * gq, cpv[gq]);
                }
                mbar_wait(&s_full[k & 1], (uint32_t)(phase0 + (k >> 1)) & 1u);
                PT_T0(t_c);
                const uint32_t S = m.part[(k & 1) * 32 + lane];
                // slack y = theta - dE: the site accepts iff y >= 0 (theta <= 2^30 and |dE| < 2^30: no overflow)
                int y = th - (int)(S - rowsum);
                PT_ACC(1, t_c);
                PT_T0(t_s);
                // The accept mask a of the block is the unique solution of the triangular system
                //   a_l = [ y_l - sum_{f<l} a_f cm[32+f][l] >= 0 ]      (cm[32+f][l] = 0 for f >= l),
                // which the site-by-site order solves by forward substitution.  Here: fixed-point iteration
                // a <- F(a) from the guess "no correction"; after t rounds the first t bits are exact, so it ends
                // after at most 33 rounds with exactly the sequential result, and in practice after two or three.
                unsigned mask = __ballot_sync(0xffffffffu, y >= 0);   // first guess: no correction at all
                int yy = y;
                if (mask | mp) {   // nothing accepted here or in block k-1: nothing to correct
                    for (int it = 0; it < 33; ++it) {
                        const unsigned mv = (mask >> (ROWS * cw)) ^ lz;
                        int part = pc;
#pragma unroll
                        for (int gq = 0; gq < RG; ++gq) part = masked_add4(part, mv, 4 * gq, cov[gq]);
                        s_xch[xb][lane][cw] = part;
                        asm volatile("bar.sync 1, %0;" ::"n"(32 * CW) : "memory");
                        if (CW == 4) {
                            const int4 pv = *reinterpret_cast<const int4*>(&s_xch[xb][lane][0]);
                            yy = y - ((pv.x + pv.y) + (pv.z + pv.w));
                        } else {
                            const int2 pv = *reinterpret_cast<const int2*>(&s_xch[xb][lane][0]);
                            yy = y - (pv.x + pv.y);
                        }
                        xb ^= 1;
                        const unsigned m2 = __ballot_sync(0xffffffffu, yy >= 0);
#ifdef PT_TIMING
                        tacc[5] += 1;
#endif
                        if (m2 == mask) break;
                        mask = m2;
                    }
                }
                PT_ACC(2, t_s);
#ifdef PT_PARANOID
                // Development builds (-DPT_PARANOID): the accept mask once more, by the forward substitution the
                // site-by-site order of Eq. 8 prescribes -- one site per step, 32 exchanges -- and compared with the
                // fixed point found above.  A mismatch raises the context's error flag (value 2): pt_sync fails.
                {
                    unsigned seq = 0u;
                    for (int l = 0; l < 32; ++l) {
                        const unsigned mv = (seq >> (ROWS * cw)) ^ lz;
                        int part = pc;
#pragma unroll
                        for (int gq = 0; gq < RG; ++gq) part = masked_add4(part, mv, 4 * gq, cov[gq]);
                        s_xch[xb][lane][cw] = part;
                        asm volatile("bar.sync 1, %0;" ::"n"(32 * CW) : "memory");
                        int ys = y;
#pragma unroll
                        for (int c2 = 0; c2 < CW; ++c2) ys -= s_xch[xb][lane][c2];
                        xb ^= 1;
                        seq |= (unsigned)__shfl_sync(0xffffffffu, ys >= 0 ? 1 : 0, l) << l;   // site l, all before it decided
                    }
                    if (seq != mask && lane == 0) *(volatile int*)d.err = 2;
                }
#endif
                if (cw == 0 && lane < 4) {
                    const uint32_t nm = expand_bits_to_nibbles(mask >> (8 * lane));
                    m.sp[wsp] = (w_old & ~nm) | (w_new & nm);
                }
                // every chain warp has read the block sums of buffer k&1 (without rounds there is no other barrier
                // between a slow warp's read and this point) before they are cleared and the buffer is handed back
                asm volatile("bar.sync 1, %0;" ::"n"(32 * CW) : "memory");
                if (cw == 0) {
                    m.part[(k & 1) * 32 + lane] = 0u;
                    __syncwarp();
                    if (lane == 0) mbar_arrive(&s_done[k & 1]);   // block k is final, buffer k&1 is free
                    if ((mask >> lane) & 1u) dE_acc += th - yy;   // yy: slack of every site at its own turn
                    n_acc += __popc(mask);
                }
                mp = mask;
                PT_ACC(0, t_c);
            }
            for (int o = 16; o > 0; o >>= 1) dE_acc += __shfl_xor_sync(0xffffffffu, dE_acc, o);
            if (owner) s_E += dE_acc;
            cta_sync();
            // a8: sample after the sweep, before the swap event (A15)
            const int nmax = direct_nmax(m.sp, W, q, s_cnt);
            if (owner) {
                oa.acc += n_acc;
                oa.att += L;
                oa.sample(s_E, nmax);
            }
            cta_sync();
            if (swap_mode == 2 && (sweep0 + s + 1) % swap_every == 0) {
                const int t_new = direct_swap_in_kernel(d, ps, e, (uint32_t)(sweep0 + s + 1), st, &s_E, event++);
                if (t_new != t) {   // the accumulators belong to the slot: hand them over when the slot changes
                    if (owner) {
                        oa.flush(d.obs + (size_t)e * d.n_rep + t);
                        oa = ObsAcc();
                    }
                    t = t_new;
                    scale = s_scale[t];
                }
            }
        }
        if (owner) {
            d.E[x] = s_E;
            if (swap_mode == 2) {
                // The observables of a slot are read-modify-written by one CTA at a time; a last counter barrier
                // orders this final flush behind the flush of whoever left the slot at an earlier event.
                asm volatile("red.release.gpu.global.add.u32 [%0], 1;" ::"l"(d.gen + e) : "memory");
                wait_arrivals(d.gen + e, (unsigned)d.n_rep * (unsigned)(event + 1), d.err);
            }
            oa.flush(d.obs + (size_t)e * d.n_rep + t);
        }
#ifdef PT_TIMING
        if (lane == 0 && d.dbg && warp < 32) {
            tacc[4] = clock64() - t_kernel;
            for (int n = 0; n < 8; ++n) d.dbg[((size_t)blockIdx.x * 32 + warp) * 8 + n] += tacc[n];
        }
#endif
    }

    cta_sync();
    for (int w = tid; w < W; w += NT) g_sp[w] = m.sp[w];
    if (swap_mode == 1) arrive_and_swap(d, e, (uint32_t)(sweep0 + n_sweeps));
    if (swap_mode == 2 && st == 0)   // all copies are identical: one CTA per ensemble writes the permutation back
        for (int t2 = tid; t2 < d.n_rep; t2 += NT) d.perm[(size_t)e * d.n_rep + t2] = s_perm[t2];
#ifdef PT_TIMING
    if (tid == 0 && d.dbg) {   // per CTA: [31][0] first start, [31][1] last end, [31][2] sum of (end - start), [31][3] launches
        unsigned long long gt_end;
        asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(gt_end));
        long long* g = d.dbg + ((size_t)blockIdx.x * 32 + 31) * 8;
        if (g[3] == 0) g[0] = (long long)gt_start;
        g[1] = (long long)gt_end;
        g[2] += (long long)(gt_end - gt_start);
        g[3] += 1;
    }
#endif
}

// ---------------------------------------------------------------------------
// a6. Total energy with the bulk machinery (Eq. 2 in reading A1):
//   E = -(1/2) sum_i S_i,   S_i = sum_j Jq[(i-j) mod L] [c_j == c_i]      (Jq[0] = 0 drops j == i).
// Same thread mapping as BULK (4 sites x 64 j per thread, couplings in registers, both 16-bit halves), the
// per-site table is the one-hot byte table of the site's own colour.  One CTA per replica (storage order).
// ---------------------------------------------------------------------------
template <bool Q16>
__global__ void __launch_bounds__(ENERGY_MAX_THREADS, 1)
energy_direct_kernel(Dev d, long long* __restrict__ E_out) {
    extern __shared__ uint32_t smem_ed[];
    uint32_t* sp = smem_ed;   // [W]
    __shared__ unsigned long long s_tot[ENERGY_MAX_THREADS / 32];
    const int L = d.L, W = d.W;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, NT = blockDim.x;
    const int g = tid & 7, jr = tid >> 3;
    const int par = g & 1, gbase = 8 * (g >> 1) + par;
    const int NJR = L / 64, NB = L >> 5;
    const bool active = jr < NJR;
    uint32_t PL[ENERGY_NPAIR], PH[ENERGY_NPAIR];
    {
        const int H = L / 2;
        const int R0 = ((gbase + 6 - 64 * jr) % L + L) % L;
        const uint32_t* lo = d.Jpair + (size_t)(2 * par) * H;
        const uint32_t* hi = lo + H;
        int r = R0;
#pragma unroll
        for (int tt = 0; tt < ENERGY_NPAIR; ++tt) {
            const int mm = (r - par) >> 1;
            PL[tt] = active ? __ldg(lo + mm) : 0u;
            PH[tt] = active ? __ldg(hi + mm) : 0u;
            r -= 2;
            r += r < 0 ? L : 0;
        }
    }
    const uint32_t* g_sp = d.spins + (size_t)blockIdx.x * W;
    for (int w = tid; w < W; w += NT) sp[w] = g_sp[w];
    __syncthreads();
    unsigned long long tot = 0ull;
    if (active) {
        int wj = 8 * jr;
        for (int kb = 0; kb < NB; ++kb) {
            int wj2 = wj + 4;
            wj2 -= wj2 >= W ? W : 0;
            const uint4 wa = *reinterpret_cast<const uint4*>(sp + wj);
            const uint4 wb = *reinterpret_cast<const uint4*>(sp + wj2);
            const uint32_t words[8] = {wa.x, wa.y, wa.z, wa.w, wb.x, wb.y, wb.z, wb.w};
            uint2 lt[4], ltb[4];
#pragma unroll
            for (int mm = 0; mm < 4; ++mm) {   // byte k of the table = [k == c_i], colours 0..7 | 8..15
                const int ci = get_nibble(sp, (kb << 5) + gbase + 2 * mm);
                const unsigned long long ta = ci < 8 ? 1ull << (8 * ci) : 0ull;
                const unsigned long long tb = ci < 8 ? 0ull : 1ull << (8 * (ci - 8));
                lt[mm] = make_uint2((uint32_t)ta, (uint32_t)(ta >> 32));
                ltb[mm] = make_uint2((uint32_t)tb, (uint32_t)(tb >> 32));
            }
            uint32_t alo[4] = {0u, 0u, 0u, 0u}, alo2[4] = {0u, 0u, 0u, 0u}, ahi[4] = {0u, 0u, 0u, 0u},
                     ahi2[4] = {0u, 0u, 0u, 0u};
#pragma unroll
            for (int u = 0; u < 16; ++u) {
                const uint32_t sel = (u & 1) ? (words[u >> 1] >> 16) : words[u >> 1];
                const uint32_t selx = sel ^ 0x8888u;
#pragma unroll
                for (int mm = 0; mm < 4; ++mm) {
                    const uint32_t S = tab_lookup<Q16>(lt[mm], ltb[mm], sel, selx);
                    const int tt = 3 - mm + 2 * u;
                    alo[mm] = __dp2a_lo(PL[tt], S, alo[mm]);
                    alo2[mm] = __dp2a_hi(PL[tt + 1], S, alo2[mm]);
                    ahi[mm] = __dp2a_lo(PH[tt], S, ahi[mm]);
                    ahi2[mm] = __dp2a_hi(PH[tt + 1], S, ahi2[mm]);
                }
            }
#pragma unroll
            for (int mm = 0; mm < 4; ++mm)
                tot += (unsigned long long)(alo[mm] + alo2[mm]) + ((unsigned long long)(ahi[mm] + ahi2[mm]) << 16);
            wj += 4;
            wj -= wj >= W ? W : 0;
        }
    }
    for (int o = 16; o > 0; o >>= 1) tot += __shfl_xor_sync(0xffffffffu, tot, o);
    if (lane == 0) s_tot[warp] = tot;
    __syncthreads();
    if (tid == 0) {
        unsigned long long t2 = 0ull;
        for (int k = 0; k < (NT >> 5); ++k) t2 += s_tot[k];
        E_out[blockIdx.x] = -(long long)(t2 / 2ull);   // the ordered-pair sum is even
    }
}

inline int launch_energy_direct(const Dev& d, long long* E_out, cudaStream_t stream) {
    if (d.q > 8)
        energy_direct_kernel<true><<<d.n_ens * d.n_rep, energy_threads(d.L), (size_t)d.W * 4, stream>>>(d, E_out);
    else
        energy_direct_kernel<false><<<d.n_ens * d.n_rep, energy_threads(d.L), (size_t)d.W * 4, stream>>>(d, E_out);
    return (int)cudaGetLastError();
}

typedef void (*direct_kernel_t)(Dev, long long, int, int, int, int);

// r_hi = largest r <= L/2 with Jq[r] >= 2^16 (0 if none).
// minb = 1: up to 168 registers per thread (fastest block sums); minb = 2: 80 registers, twice the CTAs per SM.
// wide4: a window wider than 96 sites may take four near quads per thread (else: both halves everywhere).
inline direct_kernel_t direct_kernel_variant(const Dev& d, int r_hi, int minb, bool wide4 = true) {
#ifdef PT_ONLY_HEADLINE   // development builds: only the configs[3] instantiation (fast to compile)
    return d.far ? sweep_direct_kernel<1, true, false, 1, true> : sweep_direct_kernel<1, true, false, 1>;
#else
    const bool l4096 = d.L == 4096;
    int nq = direct_nearq(d.L, r_hi);
    if (nq && direct_near_off(r_hi) > 96) {   // the wide windows: their own instantiations
        const bool big = d.L > 64 * (DIRECT_MAX_BULK / 4);
        if (big && nq == 1)
            return d.q <= 8 ? sweep_direct_kernel<1, false, false, 3, false, true> : sweep_direct_kernel<1, false, true, 3, false, true>;
        if (big && nq == 2)
            return d.q <= 8 ? sweep_direct_kernel<2, false, false, 3, false, true> : sweep_direct_kernel<2, false, true, 3, false, true>;
        if (!big && minb == 1 && nq == 2)
            return d.q <= 8 ? sweep_direct_kernel<2, false, false, 1, false, true> : sweep_direct_kernel<2, false, true, 1, false, true>;
        if (!big && minb == 1 && nq == 4 && wide4)
            return d.q <= 8 ? sweep_direct_kernel<4, false, false, 1, false, true> : sweep_direct_kernel<4, false, true, 1, false, true>;
        if (!big && minb == 4 && nq == 4 && wide4)
            return d.q <= 8 ? sweep_direct_kernel<4, false, false, 4, false, true> : sweep_direct_kernel<4, false, true, 4, false, true>;
        nq = 0;   // no instantiation for this combination: both halves everywhere
    }
    if (d.L > 64 * (DIRECT_MAX_BULK / 4)) {   // more than 64 j-ranges: every near quad has a thread of its own
        if (d.q <= 8) return nq == 1 ? sweep_direct_kernel<1, false, false, 3> : sweep_direct_kernel<0, false, false, 3>;
        return nq == 1 ? sweep_direct_kernel<1, false, true, 3> : sweep_direct_kernel<0, false, true, 3>;
    }
    if (minb == 4) {   // 128 registers, two CTAs of at most DIRECT_MID_THREADS threads per SM (nq is 2 or 4 for these L)
        if (d.q <= 8)
            return nq == 2 ? sweep_direct_kernel<2, false, false, 4>
                 : nq == 4 ? sweep_direct_kernel<4, false, false, 4> : sweep_direct_kernel<0, false, false, 4>;
        return nq == 2 ? sweep_direct_kernel<2, false, true, 4>
             : nq == 4 ? sweep_direct_kernel<4, false, true, 4> : sweep_direct_kernel<0, false, true, 4>;
    }
    if (d.q <= 8) {
        if (minb == 1) {
            switch (nq) {
                case 1:
                    if (l4096 && !d.far && getenv("PT_CW") && getenv("PT_CW")[0] == '2')   // experiment: two chain warps
                        return sweep_direct_kernel<1, true, false, 1, false, false, 2>;
                    return l4096 ? (d.far ? sweep_direct_kernel<1, true, false, 1, true> : sweep_direct_kernel<1, true, false, 1>)
                                 : sweep_direct_kernel<1, false, false, 1>;
                case 2: return sweep_direct_kernel<2, false, false, 1>;
                case 4: return sweep_direct_kernel<4, false, false, 1>;
                default: return l4096 ? sweep_direct_kernel<0, true, false, 1> : sweep_direct_kernel<0, false, false, 1>;
            }
        }
        return nq == 4 ? sweep_direct_kernel<4, false, false, 2> : sweep_direct_kernel<0, false, false, 2>;
    }
    if (minb == 1) {
        switch (nq) {
            case 1: return sweep_direct_kernel<1, false, true, 1>;
            case 2: return sweep_direct_kernel<2, false, true, 1>;
            case 4: return sweep_direct_kernel<4, false, true, 1>;
            default: return sweep_direct_kernel<0, false, true, 1>;
        }
    }
    return nq == 4 ? sweep_direct_kernel<4, false, true, 2> : sweep_direct_kernel<0, false, true, 2>;
#endif
}

// Near quads per thread of the instantiation direct_kernel_variant(d, r_hi, minb, wide4) returns (0: both halves
// everywhere): not every (window, quads, build) combination has an instantiation.  For pt_describe.
inline int direct_effective_nearq(const Dev& d, int r_hi, int minb, bool wide4) {
    const int nq = direct_nearq(d.L, r_hi);
    const bool big = d.L > 64 * (DIRECT_MAX_BULK / 4);
    if (nq && direct_near_off(r_hi) > 96) {
        if (big) return nq <= 2 ? nq : 0;
        if (minb == 1) return nq == 2 || (nq == 4 && wide4) ? nq : 0;
        if (minb == 4) return nq == 4 && wide4 ? nq : 0;
        return 0;
    }
    if (big) return nq == 1 ? 1 : 0;
    if (minb == 4) return nq == 2 || nq == 4 ? nq : 0;
    if (minb == 1) return nq == 1 || nq == 2 || nq == 4 ? nq : 0;
    return nq == 4 ? 4 : 0;
}

// Chain warps of a kernel variant (its block size is direct_threads(L, cw)).
inline int direct_chain_warps_of(direct_kernel_t k) {
    const direct_kernel_t two[] = {sweep_direct_kernel<1, true, false, 1, false, false, 2>};
    for (direct_kernel_t t : two)
        if (k == t) return 2;
    return DIRECT_CHAIN_WARPS;
}

// CTAs of a sweep kernel variant that can be resident on the device at once (0 on error).
inline int direct_coresident(direct_kernel_t kern, const Dev& d, int device) {
    const size_t smem = direct_smem_bytes(d.L, d.q);
    if (allow_max_dynamic_smem((const void*)kern, DIRECT_STATIC_SMEM) != 0) return 0;
    int per_sm = 0, n_sm = 0, coop = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, direct_threads(d.L, direct_chain_warps_of(kern)), smem) != cudaSuccess) return 0;
    if (cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, device) != cudaSuccess) return 0;
    if (cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, device) != cudaSuccess || !coop) return 0;
    return per_sm * n_sm;
}

// The kernel a context uses, and how many of its CTAs fit on the device at once (a persistent launch, swap_mode 2,
// needs all n_ens * n_rep of them).  Three register allocations of the same code: MINB = 1 (up to 168 registers, one
// CTA per SM at L >= 1088), MINB = 2 (80 registers), MINB = 4 (128 registers, two CTAs of at most 256 threads per SM:
// 1024 < L <= 2048).  The 168-register build while all replicas fit in one wave of it.  Beyond one wave:
//  * L <= 1024: the 80-register build (co-resident or not: measured 5-13 % faster at L = 256..1024 with 600..1200
//    replicas, equal at L = 1024 with 740, 2.5 % slower with 1200, profiles/r1_g_paper_shapes.md);
//  * 1024 < L <= 2048: whichever of the three has the lowest  waves x (time of a wave),  waves = ceil(replicas / CTAs
//    resident at once), with the wave times measured at L = 1088, 1536, 2048 with 32..1200 replicas
//    (profiles/r2_f_two_ctas_per_sm.md): 1 : 1.3-1.5 : 2.55 for 1, 2 and 3 CTAs per SM -- two CTAs of 128 registers
//    share an SM at 1.3x the time of one (at L = 2048 a CTA has one bulk warp per sub-partition and a block takes
//    3.5x the clocks of its IDP.2A stream, so a second CTA fills the gaps): 0.163 against 0.191 ms per sweep at
//    L = 2048 with 400 replicas, 0.434 against 0.544 with 1200; the 80-register build is a factor 1.5 slower at
//    L = 2048 and never picked there;
//  * L > 2048: the 168-register build (the 80-register one: a factor 2 slower at L = 4096).
// A context of fewer than a third of the SMs in CTAs (one of the 40 handles of configs[4]) shares the GPU with others:
// at 1024 < L <= 2048 it takes the 128-register build where that costs a lone context nothing (low-half bulk sums,
// q <= 8: 0.0738 against 0.0745 ms at L = 2048 with 32 replicas), so that two of them fit on an SM.
// PT_MINB=1|2|4 (experiments) forces the 168-, for L <= 4096 the 80-, for 1024 < L <= 2048 the 128-register build.
inline direct_kernel_t select_direct_kernel(const Dev& d, int r_hi, int device, int* coresident) {
    direct_kernel_t k1 = direct_kernel_variant(d, r_hi, 1);
    int c1 = direct_coresident(k1, d, device);
    const char* env = getenv("PT_MINB");
    const bool force1 = env && env[0] == '1';
    const bool force2 = env && env[0] == '2' && d.L <= 64 * (DIRECT_MAX_BULK / 4);
    const bool mid = direct_threads(d.L) <= DIRECT_MID_THREADS && direct_threads(d.L) > 192;   // 1024 < L <= 2048
    const bool force4 = env && env[0] == '4' && mid;
    const int R = d.n_ens * d.n_rep;
    int n_sm = 0;
    if (cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, device) != cudaSuccess) n_sm = 0;
    // One wave at L <= 2048 (one bulk warp per sub-partition): a block's time is the latency of the bulk -> chain
    // hand-off, not the instruction count.  Four near quads per thread for a wide window lengthen the tail of every
    // block and the set-up of every launch: measured equal to both halves everywhere for a lone context (0.0722
    // against 0.0730 ms at L = 2048, q = 5, sigma = 0.2, 32 replicas) and 2 % slower on configs[4]; with several
    // waves (two CTAs per SM, issue-bound) 13 % faster (0.178 against 0.204 ms at L = 2048, sigma = 0.2, 400 replicas).
    if (R <= c1 && d.L <= 2048) {
        k1 = direct_kernel_variant(d, r_hi, 1, false);
        c1 = direct_coresident(k1, d, device);   // (also sets the kernel's shared-memory attribute)
    }
    if (force1 || c1 <= 0) {
    } else if (force2) {
        k1 = direct_kernel_variant(d, r_hi, 2);
        c1 = direct_coresident(k1, d, device);
    } else if (force4) {
        k1 = direct_kernel_variant(d, r_hi, 4);
        c1 = direct_coresident(k1, d, device);
    } else if (mid) {
        const int nq = direct_nearq(d.L, r_hi);
        if (R > c1) {
            const double w4 = (d.q <= 8 && nq == 2) ? 1.3 : (d.q <= 8 && nq == 4) ? 1.4 : 1.5, w2 = 2.55;
            direct_kernel_t k4 = direct_kernel_variant(d, r_hi, 4);
            const int c4 = direct_coresident(k4, d, device);
            double best = (double)((R + c1 - 1) / c1);
            direct_kernel_t kb = k1;
            int cb = c1;
            if (c4 > c1 && w4 * ((R + c4 - 1) / c4) < best) { best = w4 * ((R + c4 - 1) / c4); kb = k4; cb = c4; }
            if (d.L < 2048) {
                direct_kernel_t k2 = direct_kernel_variant(d, r_hi, 2);
                const int c2 = direct_coresident(k2, d, device);
                if (c2 > c1 && w2 * ((R + c2 - 1) / c2) < best) { best = w2 * ((R + c2 - 1) / c2); kb = k2; cb = c2; }
            }
            k1 = kb;
            c1 = cb;
        } else if (3 * R < n_sm && d.q <= 8 && nq == 2) {   // (q > 8 at 128 registers: 22 % slower alone, 2 % slower on configs[4])
            direct_kernel_t k4 = direct_kernel_variant(d, r_hi, 4);
            const int c4 = direct_coresident(k4, d, device);
            if (c4 > c1) { k1 = k4; c1 = c4; }
        }
    } else if (R > c1 && d.L < 2048) {
        direct_kernel_t k2 = direct_kernel_variant(d, r_hi, 2);
        const int c2 = direct_coresident(k2, d, device);
        if (c2 > c1) { k1 = k2; c1 = c2; }
    }
    if (coresident) *coresident = c1;
    return k1;
}

// Returns a cudaError_t as int.  swap_mode 0/1: one ordinary launch of n_sweeps sweeps, optionally closed by a swap
// event.  swap_mode 2: cooperative (all CTAs co-resident) persistent launch with the swap events inside the kernel.
// (Programmatic dependent launch was tried for swap_mode 1 and removed: streams with thousands of dependent
// launches of this kernel queued back to back occasionally never finished on this driver, and for the small
// contexts that still use swap_mode 1 it was slower than ordinary launches: 0.41-0.48 s against 0.39 s for 10000
// sweeps of configs[2].)
inline int launch_sweep_direct(direct_kernel_t kern, const Dev& d, long long sweep0, int n_sweeps, int swap_mode,
                               int swap_every, int r_hi, cudaStream_t stream) {
    const size_t smem = direct_smem_bytes(d.L, d.q);
    cudaError_t err = cudaSuccess;   // (the shared-memory attribute was set once, in direct_coresident)
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)(swap_mode == 3 ? d.n_local : d.n_ens * d.n_rep));
    cfg.blockDim = dim3((unsigned)direct_threads(d.L, direct_chain_warps_of(kern)));
    cfg.dynamicSmemBytes = smem;
    cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    if (swap_mode == 2) {
        attr[0].id = cudaLaunchAttributeCooperative;
        attr[0].val.cooperative = 1;
    }
    cfg.attrs = attr;
    cfg.numAttrs = swap_mode == 2 ? 1 : 0;
    err = cudaLaunchKernelEx(&cfg, kern, d, sweep0, n_sweeps, swap_mode, swap_every, r_hi);
    if (err != cudaSuccess) return (int)err;
    return (int)cudaGetLastError();
}

}  // namespace ptk

// pt_kernels.cuh -- set-up, energy, swap and I/O kernels of libpt (sm_100a).
// The sweep kernels are in pt_sweep_field.cuh and pt_sweep_direct.cuh.
#pragma once
#include <cstdint>
#include <mutex>
#include <set>
#include <utility>

#include "pt.h"
#include "pt_device.cuh"

namespace ptk {

using namespace ptdev;

// Opt a kernel in to the full dynamic shared memory of an SM once per process and device (not per launch: the
// attribute belongs to the function, and contexts of different L share functions and may launch from different
// host threads).  Returns a cudaError_t as int.
inline int allow_max_dynamic_smem(const void* kernel, int static_bytes) {
    static std::mutex mu;
    static std::set<std::pair<const void*, int>> done;
    int dev = 0;
    cudaError_t err = cudaGetDevice(&dev);
    if (err != cudaSuccess) return (int)err;
    std::lock_guard<std::mutex> lock(mu);
    if (done.count({kernel, dev})) return 0;
    err = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024 - static_bytes);
    if (err == cudaSuccess) done.insert({kernel, dev});
    return (int)err;
}

// Everything a kernel needs to know about a context (passed by value).  New fields go at the END: ptxas' schedule of
// sweep_direct_kernel changes with the layout of its parameters (a field inserted after ens_base cost the headline
// workload 3 %, measured A/B on one GPU; appended, the SASS is the same up to constant-bank offsets).
// Parameters and buffers of the helper CTAs of a persistent launch (pt_sweep_direct.cuh, HELPERS), in device memory.
struct HelpDev {
    int n_help;               // CTAs beyond the n_rep sweep CTAs: they sum part of the pair terms of other replicas
    int help_cap;             // block tasks per helper and sweep
    int help_end;             // blocks help_k0 .. help_end - 1 of a sweep can be served
    int help_k0;              // first block of a sweep that can be served
    int help_whot;            // weight of a hot slot in the split of a helper's capacity (a cold slot: 1)
    unsigned long long* hs;   // [n_rep][L] helper block sums by storage index and site: sum | stamp << 32
    int* Apub;                // [2][n_rep] accepted changes of the sweep, published with Epub
    uint32_t* spub;           // [2][n_rep][W] spins as decided, by sweep parity and storage index
    unsigned* mprog;          // [n_rep] decided blocks in units of 16 (launch-local, monotone), by storage index
};

struct Dev {
    int L, W, q, n_ens, n_rep, ens_base;
    int rep_base, n_local;    // slot-sharded contexts (pt_create_shard): this process sweeps the configurations with
                              // storage index rep_base .. rep_base + n_local - 1; otherwise 0, n_rep
    int count_swaps;          // 0: this shard leaves the swap counters to the shard with rep_base = 0
    uint32_t key0, key1;
    uint32_t rowsum;          // sum_r Jq[r] (< 2^31)
    const int32_t* Jq;        // [L]
    const uint32_t* Jpair;    // direct variant: [4][L/2] packed 16-bit halves, see pack_pairs_kernel
    const double* beta;       // [n_rep]
    const double* thr_scale;  // [n_rep] 2^24/beta
    uint32_t* spins;          // [n_ens*n_rep][W]   storage order
    long long* E;             // [n_ens*n_rep]      storage order
    int* perm;                // [n_ens][n_rep]     slot -> storage index inside the ensemble
    pt_obs* obs;              // [n_ens][n_rep]     slot order
    int32_t* h;               // [n_ens*n_rep][q][L] storage order (field variant)
    unsigned* done;           // [n_ens] arrival counters of the swap event
    unsigned* gen;            // [n_ens] arrivals at the swap events of the running persistent launch
    long long* Epub;          // [2][n_ens][n_rep] energies published for those events, by storage index
    int* err;                 // raised by a kernel whose in-kernel barrier timed out (host-mapped: read by pt_sync)
    long long* dbg;           // PT_TIMING builds: [n_ens*n_rep][32 warps][8] clock sums (else unused)
    int bits;                 // bits per spin in spins[]: 4 (q <= 16, 8 sites per word) or 8 (q <= 64, 4 sites per word)
    int far;                  // direct variant, L = 4096: the couplings of every far j-range (jr = 16..47) lie within 255 of
                              // their minimum, which is < 2^15 (pt_sweep_direct.cuh, FAR); at the end of the struct: the
                              // order of the kernel parameters changes the schedule of the sweep kernel
    const struct HelpDev* hlp; // helper CTAs of a persistent launch (pt_sweep_direct.cuh, HELPERS), else nullptr.  One pointer at
                              // the end of the struct: more kernel parameters change the schedule of the sweep kernel
};

// ---------------------------------------------------------------------------
// a1. J* table (Eqs. 5-7).  With x = r/L and s = 1+sigma,
//   J*(r) = sum_n |r+nL|^-s = L^-s [ zeta(s,x) + zeta(s,1-x) ],
// zeta(s,y) = sum_{k>=0} (k+y)^-s the Hurwitz zeta function of Eq. 7 (Eq. 6
// is the same expression with the k = 0 term of zeta(s,x) written as r^-s).
// Each zeta is summed directly for k < NDIRECT and closed with the
// Euler-Maclaurin remainder at y + NDIRECT.  One thread per r <= L/2; the
// table is mirrored so that it is exactly symmetric (A3); Jq[0] = 0 (A2).
// ---------------------------------------------------------------------------
__device__ inline double zeta_tail(double s, double y) {
    // sum_{k>=0} (y+k)^-s for y >= 16:  y^(1-s)/(s-1) + y^-s/2 + sum_m B_2m/(2m)! s^(2m-1) y^(-s-2m+1)
    const double ys = pow(y, -s);
    const double iy2 = 1.0 / (y * y);
    double term = s * ys / y;  // s y^(-s-1)
    double acc = 0.0;
    const double b[6] = {1.0 / 12.0, -1.0 / 720.0, 1.0 / 30240.0, -1.0 / 1209600.0, 1.0 / 47900160.0,
                         -691.0 / 1307674368000.0};
    double corr[6];
#pragma unroll
    for (int m = 0; m < 6; ++m) {
        corr[m] = b[m] * term;
        term *= (s + (2 * m + 1)) * (s + (2 * m + 2)) * iy2;
    }
#pragma unroll
    for (int m = 5; m >= 0; --m) acc += corr[m];
    return acc + 0.5 * ys + ys * y / (s - 1.0);
}

__global__ void jstar_kernel(int L, double sigma, int32_t* __restrict__ Jq, double* __restrict__ Jreal) {
    const int r = blockIdx.x * blockDim.x + threadIdx.x;
    if (r == 0) { Jq[0] = 0; if (Jreal) Jreal[0] = 0.0; }
    if (r < 1 || r > L / 2) return;
    constexpr int NDIRECT = 16;
    const double s = 1.0 + sigma;
    const double x = (double)r / (double)L;
    double acc = zeta_tail(s, NDIRECT + x) + zeta_tail(s, NDIRECT + 1.0 - x);
    for (int k = NDIRECT - 1; k >= 0; --k) acc += pow(k + x, -s) + pow(k + 1.0 - x, -s);
    const double J = acc * pow((double)L, -s);
    const long long v = __double2ll_rn(J * 16777216.0);  // scale 2^24 (A16), ties to even
    Jq[r] = (int32_t)v;
    Jq[L - r] = (int32_t)v;
    if (Jreal) { Jreal[r] = J; Jreal[L - r] = J; }
}

// Direct variant tables.  For parity p in {0,1} and m in [0, L/2): r = 2m+p,
//   lo[p][m] = (Jq[r] & 0xffff) | (Jq[r-1] & 0xffff) << 16
//   hi[p][m] = (Jq[r] >> 16)    | (Jq[r-1] >> 16)    << 16       (indices mod L)
// laid out as Jpair[0]=lo[0], [1]=hi[0], [2]=lo[1], [3]=hi[1], each L/2 words.
__global__ void pack_pairs_kernel(int L, const int32_t* __restrict__ Jq, uint32_t* __restrict__ Jpair) {
    const int m = blockIdx.x * blockDim.x + threadIdx.x;
    const int H = L / 2;
    if (m >= H) return;
    for (int p = 0; p < 2; ++p) {
        const int r = 2 * m + p;
        const uint32_t j0 = (uint32_t)Jq[r], j1 = (uint32_t)Jq[(r + L - 1) % L];
        Jpair[(2 * p + 0) * H + m] = (j0 & 0xffffu) | ((j1 & 0xffffu) << 16);
        Jpair[(2 * p + 1) * H + m] = (j0 >> 16) | ((j1 >> 16) << 16);
    }
}

// ---------------------------------------------------------------------------
// a2. Hot start (configs; not in the paper): colour of site i of slot t of
// ensemble e = mulhi32(Philox(i, 0, t, e<<4|INIT).w0, q).  One thread per word.
// ---------------------------------------------------------------------------
__global__ void init_spins_kernel(Dev d) {
    const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long total = (long long)d.n_ens * d.n_rep * d.W;
    if (gid >= total) return;
    const int w = (int)(gid % d.W);
    const int x = (int)(gid / d.W);
    const int e = x / d.n_rep, t = x % d.n_rep;
    const uint32_t c3 = ((uint32_t)(d.ens_base + e) << 4) | TAG_INIT;
    uint32_t word = 0;
    const int per = 32 / d.bits;
    for (int n = 0; n < per; ++n) {
        const Philox4 p = philox4x32_10((uint32_t)(per * w + n), 0u, (uint32_t)t, c3, d.key0, d.key1);
        word |= __umulhi(p.w0, (uint32_t)d.q) << (d.bits * n);
    }
    d.spins[gid] = word;  // storage index == slot at creation (perm = identity)
}

__global__ void init_perm_kernel(Dev d) {
    const int gid = blockIdx.x * blockDim.x + threadIdx.x;
    if (gid < d.n_ens * d.n_rep) d.perm[gid] = gid % d.n_rep;
}

// ---------------------------------------------------------------------------
// a6. Total energy (Eq. 2 in reading A1):
//   E = -sum_{i<j} Jq[j-i] [c_i==c_j] = -(1/2) sum_i sum_{j!=i} Jq[|i-j|] [c_j==c_i].
// One CTA per replica (storage order), one site per thread and pass; spins and
// couplings staged in shared memory; SWAR match of the 8 (or 4) sites of a word.
// dynamic smem: (L + W) * 4 bytes.
// ---------------------------------------------------------------------------
__global__ void __launch_bounds__(256) energy_kernel(Dev d, long long* __restrict__ E_out) {
    extern __shared__ uint32_t smem_e[];
    int32_t* J = (int32_t*)smem_e;
    uint32_t* sp = smem_e + d.L;
    __shared__ long long s_part[8];
    const int x = blockIdx.x;
    for (int r = threadIdx.x; r < d.L; r += blockDim.x) J[r] = d.Jq[r];
    for (int w = threadIdx.x; w < d.W; w += blockDim.x) sp[w] = d.spins[(size_t)x * d.W + w];
    __syncthreads();
    long long acc = 0;
    const int per = 32 / d.bits, lg = d.bits == 4 ? 2 : 3;
    for (int i = threadIdx.x; i < d.L; i += blockDim.x) {
        const uint32_t a = (uint32_t)get_colour(sp, i, d.bits);
        long long row = 0;
        for (int w = 0; w < d.W; ++w) {
            uint32_t m = match_colours(sp[w], a, d.bits);
            while (m) {
                const int bit = __ffs(m) - 1;
                m &= m - 1;
                const int j = per * w + (bit >> lg);
                const int dist = j > i ? j - i : i - j;
                row += J[dist];  // J[0] = 0 removes j == i
            }
        }
        acc += row;
    }
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    if ((threadIdx.x & 31) == 0) s_part[threadIdx.x >> 5] = acc;
    __syncthreads();
    if (threadIdx.x == 0) {
        long long tot = 0;
        for (int k = 0; k < (int)(blockDim.x >> 5); ++k) tot += s_part[k];
        E_out[x] = -(tot / 2);  // the ordered-pair sum is even
    }
}

// ---------------------------------------------------------------------------
// Local fields of the field variant (north_star (3)):
//   h[x][k][i] = sum_{j!=i} Jq[|i-j|] [c_j==k].   One CTA per replica.
// dynamic smem: (L + W) * 4 bytes.
// ---------------------------------------------------------------------------
__global__ void __launch_bounds__(256) build_fields_kernel(Dev d) {
    extern __shared__ uint32_t smem_e[];
    int32_t* J = (int32_t*)smem_e;
    uint32_t* sp = smem_e + d.L;
    const int x = blockIdx.x;
    for (int r = threadIdx.x; r < d.L; r += blockDim.x) J[r] = d.Jq[r];
    for (int w = threadIdx.x; w < d.W; w += blockDim.x) sp[w] = d.spins[(size_t)x * d.W + w];
    __syncthreads();
    int32_t* hx = d.h + (size_t)x * d.q * d.L;
    const int per = 32 / d.bits, lg = d.bits == 4 ? 2 : 3;
    for (int i = threadIdx.x; i < d.L; i += blockDim.x) {
        for (int k = 0; k < d.q; ++k) {
            int32_t acc = 0;
            for (int w = 0; w < d.W; ++w) {
                uint32_t m = match_colours(sp[w], (uint32_t)k, d.bits);
                while (m) {
                    const int bit = __ffs(m) - 1;
                    m &= m - 1;
                    const int j = per * w + (bit >> lg);
                    const int dist = j > i ? j - i : i - j;
                    acc += J[dist];
                }
            }
            hx[(size_t)k * d.L + i] = acc;
        }
    }
}

// ---------------------------------------------------------------------------
// a7. Swap event (Eq. 9; 126: pairs (t,t+1), t even, then t
// odd).  Run by ONE CTA per ensemble after every replica of the ensemble has
// published its energy.  Configurations stay where they are stored; the
// slot -> storage permutation is exchanged (A12).  Accept iff
//   d = (beta_t - beta_{t+1}) (E_t - E_{t+1}) 2^-24 >= 0  or  u < exp(d),
// u from Philox(t, sweep, 0, e<<4|SWAP).  fp64 throughout, one rounding in d.
// ---------------------------------------------------------------------------
// All global reads of state that another CTA may have written go to L2 (__ldcg / atomics): inside a persistent
// launch the event is run by a different CTA every time and L1 is not coherent.
__device__ inline void swap_event(const Dev& d, int e, uint32_t sweep) {
    int* perm = d.perm + (size_t)e * d.n_rep;
    const long long* E = d.E + (size_t)e * d.n_rep;
    pt_obs* obs = d.obs + (size_t)e * d.n_rep;
    const uint32_t c3 = ((uint32_t)(d.ens_base + e) << 4) | TAG_SWAP;
    for (int stage = 0; stage < 2; ++stage) {
        for (int t = stage + 2 * (int)threadIdx.x; t + 1 < d.n_rep; t += 2 * (int)blockDim.x) {
            const int sa = __ldcg(perm + t), sb = __ldcg(perm + t + 1);
            const long long Ea = __ldcg(E + sa), Eb = __ldcg(E + sb);
            const double dd = __dmul_rn(d.beta[t] - d.beta[t + 1], ldexp((double)(Ea - Eb), -24));
            const Philox4 p = philox4x32_10((uint32_t)t, sweep, 0u, c3, d.key0, d.key1);
            const double u = uniform53(p.w1, p.w2);
            if (d.count_swaps) atomicAdd((unsigned long long*)&obs[t].swap_attempts, 1ull);
            if (dd >= 0.0 || u < exp(dd)) {
                __stcg(perm + t, sb);
                __stcg(perm + t + 1, sa);
                if (d.count_swaps) atomicAdd((unsigned long long*)&obs[t].swap_accepts, 1ull);
            }
        }
        __threadfence_block();
        asm volatile("bar.sync 0;" ::: "memory");   // all threads of the CTA, also from role-specialised code
    }
}

// Called by every CTA of a sweep kernel at the end of a launch that ends with a
// swap event: the CTA that arrives last at the ensemble's counter runs the
// event (no CTA ever waits for another one).  All threads of the CTA must call.
__device__ inline void arrive_and_swap(const Dev& d, int e, uint32_t sweep) {
    __shared__ int s_last;
    __threadfence();  // this thread's global writes (E, spins, fields, obs) before the arrival
    __syncthreads();
    if (threadIdx.x == 0) {
        const unsigned prev = atomicAdd(d.done + e, 1u);
        s_last = (prev == (unsigned)d.n_rep - 1u);
        __threadfence();
    }
    __syncthreads();
    if (s_last) {
        swap_event(d, e, sweep);
        if (threadIdx.x == 0) d.done[e] = 0u;
    }
}

// Stand-alone swap kernel (one CTA per ensemble), used when a swap event has
// to follow sweeps that were launched without one.
__global__ void swap_kernel(Dev d, uint32_t sweep) { swap_event(d, blockIdx.x, sweep); }

// ---------------------------------------------------------------------------
// a8 helper.  N_max = max_k N_k of the configuration in packed words sp[W]
// (Eq. 10).  All threads call; result valid in thread 0.
// s_cnt: PT_QMAX ints of shared memory.
// ---------------------------------------------------------------------------
constexpr int PT_QMAX = 64;
__device__ inline int count_nmax(const uint32_t* sp, int W, int q, int bits, int* s_cnt) {
    if (threadIdx.x < PT_QMAX) s_cnt[threadIdx.x] = 0;
    __syncthreads();
    for (int w = threadIdx.x; w < W; w += blockDim.x) {
        const uint32_t word = sp[w];
        for (int k = 0; k < q; ++k) {
            const int c = __popc(match_colours(word, (uint32_t)k, bits));
            if (c) atomicAdd(&s_cnt[k], c);
        }
    }
    __syncthreads();
    int nmax = 0;
    if (threadIdx.x == 0)
        for (int k = 0; k < q; ++k) nmax = max(nmax, s_cnt[k]);
    return nmax;
}

// Per-launch accumulators kept by thread 0 of a sweep CTA.
struct ObsAcc {
    long long n = 0, sE = 0, sN = 0, sN2 = 0, sN3 = 0, acc = 0, att = 0;
    unsigned long long e2lo = 0;
    long long e2hi = 0;
    unsigned long long e4[4] = {0, 0, 0, 0};
    unsigned long long n4lo = 0;
    long long n4hi = 0;
    __device__ void sample(long long E, int nmax) {
        const long long nm = nmax, nm2 = nm * nm;
        n += 1; sE += E; sN += nm; sN2 += nm2; sN3 += nm2 * nm;
        add_square_128(e2lo, e2hi, E);
        add_fourth_256(e4, E);
        add_square_128(n4lo, n4hi, nm2);
    }
    // Adds the accumulators to the slot's pt_obs.  One writer at a time per slot, but successive writers may be
    // different CTAs (persistent launches, ordered by the swap barrier): all loads and stores go to L2; the loads are
    // independent, so the whole flush costs one L2 round trip.  The swap counters (words 8, 9) are not touched here.
    __device__ void flush(pt_obs* o) const {
        typedef unsigned long long u64;
        // Nothing gathered (the configuration moved into this slot at the last swap event of the launch): the slot's
        // previous holder may be flushing right now, and it is the only one with something to add.
        if (n == 0 && att == 0) return;
        u64* p = (u64*)o;
        u64 v[18];
#pragma unroll
        for (int k = 0; k < 18; ++k) v[k] = (k >= 8 && k <= 10) ? 0ull : __ldcg(p + k);
        v[0] += (u64)n; v[1] += (u64)sE; v[4] += (u64)sN; v[5] += (u64)sN2; v[6] += (u64)att; v[7] += (u64)acc;
        { const u64 lo = v[2] + e2lo; v[3] += (u64)e2hi + (lo < v[2] ? 1ull : 0ull); v[2] = lo; }
        u64 carry = 0ull;
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            const u64 t = v[11 + k] + carry;
            const u64 c0 = t < carry ? 1ull : 0ull;
            const u64 u = t + e4[k];
            carry = c0 + (u < t ? 1ull : 0ull);
            v[11 + k] = u;
        }
        v[15] += (u64)sN3;
        { const u64 lo = v[16] + n4lo; v[17] += (u64)n4hi + (lo < v[16] ? 1ull : 0ull); v[16] = lo; }
#pragma unroll
        for (int k = 0; k < 18; ++k)
            if (k < 8 || k > 10) __stcg(p + k, v[k]);
    }
};
static_assert(sizeof(pt_obs) == 18 * 8, "ObsAcc::flush addresses pt_obs as 18 64-bit words");

// ---------------------------------------------------------------------------
// I/O kernels (slot order outside, storage order inside).
// ---------------------------------------------------------------------------
__global__ void unpack_spins_kernel(Dev d, uint8_t* __restrict__ out) {
    const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long total = (long long)d.n_ens * d.n_rep * d.W;
    if (gid >= total) return;
    const int w = (int)(gid % d.W);
    const int x = (int)(gid / d.W);  // e*n_rep + slot
    const int e = x / d.n_rep;
    const int st = d.perm[x];
    const uint32_t word = d.spins[((size_t)e * d.n_rep + st) * d.W + w];
    const int per = 32 / d.bits;
    const uint32_t mask = (1u << d.bits) - 1u;
    uint8_t* o = out + (size_t)x * d.L + per * w;
    for (int n = 0; n < per; ++n) o[n] = (uint8_t)(((word >> (d.bits * n)) & mask) + 1u);  // A4: API colours 1..q
}

__global__ void check_spins_kernel(Dev d, const uint8_t* __restrict__ in, int* __restrict__ bad) {
    const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long total = (long long)d.n_ens * d.n_rep * d.L;
    if (gid >= total) return;
    const int v = in[gid];
    if (v < 1 || v > d.q) atomicOr(bad, 1);
}

__global__ void pack_spins_kernel(Dev d, const uint8_t* __restrict__ in) {
    const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long total = (long long)d.n_ens * d.n_rep * d.W;
    if (gid >= total) return;
    const int w = (int)(gid % d.W);
    const int x = (int)(gid / d.W);
    const int e = x / d.n_rep;
    const int st = d.perm[x];
    const int per = 32 / d.bits;
    const uint8_t* s = in + (size_t)x * d.L + per * w;
    uint32_t word = 0;
    for (int n = 0; n < per; ++n) word |= (uint32_t)(s[n] - 1) << (d.bits * n);
    d.spins[((size_t)e * d.n_rep + st) * d.W + w] = word;
}

// out[e][slot] = in[e][perm[e][slot]]
__global__ void gather_slots_kernel(Dev d, const long long* __restrict__ in, long long* __restrict__ out) {
    const int gid = blockIdx.x * blockDim.x + threadIdx.x;
    if (gid >= d.n_ens * d.n_rep) return;
    const int e = gid / d.n_rep;
    out[gid] = in[(size_t)e * d.n_rep + d.perm[gid]];
}

// out[e][perm[e][slot]] = in[e][slot]
__global__ void scatter_slots_kernel(Dev d, const long long* __restrict__ in, long long* __restrict__ out) {
    const int gid = blockIdx.x * blockDim.x + threadIdx.x;
    if (gid >= d.n_ens * d.n_rep) return;
    const int e = gid / d.n_rep;
    out[(size_t)e * d.n_rep + d.perm[gid]] = in[gid];
}

}  // namespace ptk

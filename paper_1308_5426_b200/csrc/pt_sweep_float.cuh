// pt_sweep_float.cuh -- the paper's own arithmetic as a comparison variant.
//
// "all calculations ... in single precision ... rounding errors"; :110-124 (section 4.2): one
// thread block per replica, "each thread sums a subset of pair terms" of the energy of the flipped spin, followed by a
// parallel reduction; fp64 "about half the speed" (:216).  This kernel is that design, restated for the comparison:
// 128 threads per replica, thread t adds the terms j = t, t+128, ... in increasing j, the 128 partial sums are
// combined by a binary tree (strides 64, 32, .., 1), in T = float or double.  The model is the SAME quantised model
// as everywhere else: couplings Jf[r] = (T)(Jq[r] 2^-24), so the fp64 variant reproduces the exact integer
// trajectory (every fp64 sum of 25-bit couplings is exact) and the fp32 variant shows what single-precision sums
// cost.  Eq. 8 and Eq. 9 are evaluated in fp64 on the T values on both sides (no libm expf).  The same Philox stream
// as the integer variants.  Not a performance path: it exists to measure the paper's claims on this hardware.
#pragma once
#include "pt_kernels.cuh"

namespace ptk {

constexpr int FLOAT_THREADS = 128;

// dynamic smem: Jf[L] (T) | u[L] (double) | c[L] (uint8) | b[L] (uint8); static: the 128 partial sums
template <typename T>
__host__ __device__ inline size_t float_smem_bytes(int L) {
    return (size_t)L * (sizeof(T) + sizeof(double) + 2);
}

// Swap event on floating-point energies (Eq. 9, two stages :126): as swap_event, with
// d = (beta_t - beta_{t+1}) (E_t - E_{t+1}) in fp64 on the energies Ef (storage order, units of 1).
__device__ inline void swap_event_float(const Dev& d, const double* Ef, int e, uint32_t sweep) {
    int* perm = d.perm + (size_t)e * d.n_rep;
    const double* E = Ef + (size_t)e * d.n_rep;
    pt_obs* obs = d.obs + (size_t)e * d.n_rep;
    const uint32_t c3 = ((uint32_t)(d.ens_base + e) << 4) | TAG_SWAP;
    for (int stage = 0; stage < 2; ++stage) {
        for (int t = stage + 2 * (int)threadIdx.x; t + 1 < d.n_rep; t += 2 * (int)blockDim.x) {
            const int sa = __ldcg(perm + t), sb = __ldcg(perm + t + 1);
            const double dd = __dmul_rn(d.beta[t] - d.beta[t + 1], __ldcg(E + sa) - __ldcg(E + sb));
            const Philox4 p = philox4x32_10((uint32_t)t, sweep, 0u, c3, d.key0, d.key1);
            const double u = uniform53(p.w1, p.w2);
            atomicAdd((unsigned long long*)&obs[t].swap_attempts, 1ull);
            if (dd >= 0.0 || u < exp(dd)) {
                __stcg(perm + t, sb);
                __stcg(perm + t + 1, sa);
                atomicAdd((unsigned long long*)&obs[t].swap_accepts, 1ull);
            }
        }
        __threadfence_block();
        __syncthreads();
    }
}

template <typename T>
__global__ void __launch_bounds__(FLOAT_THREADS)
sweep_float_kernel(Dev d, double* __restrict__ Ef, long long sweep0, int n_sweeps, int do_swap) {
    extern __shared__ __align__(16) unsigned char smem_fl[];
    const int L = d.L, W = d.W, q = d.q;
    T* Jf = reinterpret_cast<T*>(smem_fl);
    double* us = reinterpret_cast<double*>(smem_fl + (size_t)L * sizeof(T));
    uint8_t* c = reinterpret_cast<uint8_t*>(us + L);
    uint8_t* bq = c + L;
    __shared__ T s_part[FLOAT_THREADS];
    __shared__ int s_cnt[PT_QMAX];
    __shared__ int s_last;

    const int tid = threadIdx.x;
    const int e = blockIdx.x / d.n_rep, t = blockIdx.x % d.n_rep;
    const int st = d.perm[blockIdx.x];
    const size_t x = (size_t)e * d.n_rep + st;
    uint32_t* g_sp = d.spins + x * W;
    for (int r = tid; r < L; r += FLOAT_THREADS) Jf[r] = (T)ldexp((double)d.Jq[r], -24);
    for (int i = tid; i < L; i += FLOAT_THREADS) c[i] = (uint8_t)get_colour(g_sp, i, d.bits);
    T E = (T)Ef[x];                       // thread 0's copy is the running energy
    const double beta = d.beta[t];
    const uint32_t c3 = ((uint32_t)(d.ens_base + e) << 4) | TAG_SWEEP;
    ObsAcc oa;
    __syncthreads();

    for (int s = 0; s < n_sweeps; ++s) {
        const uint32_t sweep = (uint32_t)(sweep0 + s + 1);
        // proposals and uniforms of all sites (A6, A7): every site is visited once, so its colour at its turn is its
        // colour now
        for (int i = tid; i < L; i += FLOAT_THREADS) {
            const Philox4 p = philox4x32_10((uint32_t)i, sweep, (uint32_t)t, c3, d.key0, d.key1);
            const uint32_t a = c[i];
            const uint32_t k = __umulhi(p.w0, (uint32_t)(q - 1));
            bq[i] = (uint8_t)(k + (k >= a ? 1u : 0u));
            us[i] = uniform53(p.w1, p.w2);
        }
        __syncthreads();
        int n_acc = 0;
        for (int i = 0; i < L; ++i) {
            const int a = c[i], b = bq[i];
            // thread-split sum of the pair terms of site i, then the tree
            T acc = (T)0;
            for (int j = tid; j < L; j += FLOAT_THREADS) {
                if (j == i) continue;
                const int dist = j > i ? j - i : i - j;
                const T J = Jf[dist];
                const int cj = c[j];
                if (cj == a) acc = acc + J;
                else if (cj == b) acc = acc - J;
            }
            s_part[tid] = acc;
            __syncthreads();
            if (tid < 64) s_part[tid] = s_part[tid] + s_part[tid + 64];
            __syncthreads();
            if (tid < 32) {
                T v = s_part[tid] + s_part[tid + 32];
#pragma unroll
                for (int o = 16; o >= 1; o >>= 1) v = v + __shfl_down_sync(0xffffffffu, v, o);
                if (tid == 0) {
                    const T dE = v;
                    bool acc_it = dE <= (T)0;
                    if (!acc_it) acc_it = us[i] < exp(-(beta * (double)dE));   // Eq. 8 in fp64 on the T value
                    if (acc_it) {
                        c[i] = (uint8_t)b;
                        E = E + dE;
                        n_acc += 1;
                    }
                }
            }
            __syncthreads();
        }
        // a8: sample after the sweep (A15); the accumulators see the running energy in fixed point
        if (tid < PT_QMAX) s_cnt[tid] = 0;
        __syncthreads();
        for (int i = tid; i < L; i += FLOAT_THREADS) atomicAdd(&s_cnt[c[i]], 1);
        __syncthreads();
        if (tid == 0) {
            int nmax = 0;
            for (int k = 0; k < q; ++k) nmax = max(nmax, s_cnt[k]);
            oa.acc += n_acc;
            oa.att += L;
            oa.sample(__double2ll_rn(ldexp((double)E, 24)), nmax);
        }
        __syncthreads();
    }

    for (int w = tid; w < W; w += FLOAT_THREADS) {
        uint32_t word = 0;
        const int per = 32 / d.bits;
        for (int n = 0; n < per; ++n) word |= (uint32_t)c[per * w + n] << (d.bits * n);
        g_sp[w] = word;
    }
    if (tid == 0) {
        Ef[x] = (double)E;
        d.E[x] = __double2ll_rn(ldexp((double)E, 24));
        oa.flush(d.obs + blockIdx.x);
    }
    if (do_swap) {   // the CTA that arrives last runs the event, then brings the fixed-point copies in line
        __threadfence();
        __syncthreads();
        if (tid == 0) {
            const unsigned prev = atomicAdd(d.done + e, 1u);
            s_last = (prev == (unsigned)d.n_rep - 1u);
            __threadfence();
        }
        __syncthreads();
        if (s_last) {
            swap_event_float(d, Ef, e, (uint32_t)(sweep0 + n_sweeps));
            if (tid == 0) d.done[e] = 0u;
        }
    }
}

// Ef[x] = (T) (E[x] 2^-24): entering a floating-point variant from exact integer energies.
template <typename T>
__global__ void energy_to_float_kernel(Dev d, double* __restrict__ Ef) {
    const int gid = blockIdx.x * blockDim.x + threadIdx.x;
    if (gid < d.n_ens * d.n_rep) Ef[gid] = (double)(T)ldexp((double)d.E[gid], -24);
}

}  // namespace ptk

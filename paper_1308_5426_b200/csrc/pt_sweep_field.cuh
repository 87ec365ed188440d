// pt_sweep_field.cuh -- Metropolis sweep, local-field variant (north_star (3)).
//
// One CTA per replica.  Shared memory holds the couplings Jq[L], the packed
// spins, the per-colour local fields h[k][i] = sum_{j!=i} Jq[|i-j|][c_j==k]
// (colour-major, so that consecutive threads update consecutive banks), and
// for the running sweep the proposed colours and integer acceptance
// thresholds of all sites.  Because the generator is counter based and every
// site is visited once per sweep, proposal b_i and threshold theta_i of every
// site are known at the start of the sweep and are drawn by all threads in
// parallel; the sequential part of Eq. 8 is then
//   dE_i = h[a_i][i] - h[b_i][i]  (energy of the changed spin
//   before and after),   accept iff dE_i <= theta_i,
// which warp 0 evaluates for 32 consecutive sites at once against the current
// fields: the first accepting lane is THE next accepted step of the sequential
// sweep (all sites before it reject against exactly these fields).  The whole
// CTA then applies it: h[a][j] -= Jq[|j-f|], h[b][j] += Jq[|j-f|] for all j,
// and the scan resumes behind it.  Results are identical to the site-by-site
// order because all arithmetic is integer.
#pragma once
#include "pt_kernels.cuh"

namespace ptk {

constexpr int FIELD_THREADS = 512;

// RANDOM (site order of reading A5': "L Metropolis steps ... an average of one Monte Carlo step per spin",
// PAPER.md:112-114): step n of a sweep visits site mulhi32(w3, L) of the Philox draw keyed by (n, sweep, slot); the
// same draw gives the proposal (w0) and the uniform (w1, w2).  A site can be visited twice in a sweep, so the old
// colour a -- and with it the proposed colour k + (k >= a) -- is read at the step's turn, not at the start of the
// sweep; the scan over 32 consecutive STEPS is otherwise the same: the first accepting step is the next change.
//
// BITS: 4 bits per spin (q <= 16, W = L/8 words) or 8 (16 < q <= 64, W = L/4 words); the arithmetic is the same.
//
// dynamic smem layout (32-bit words): J[L] | theta[L] | sp[W] | bq[W] | h[q*L]
//                            RANDOM: J[L] | theta[L] | sp[W] | site[L] | kk[L/4] | h[q*L]
__host__ __device__ inline size_t field_smem_bytes(int L, int q, bool random_order = false) {
    const int W = q <= 16 ? L / 8 : L / 4;
    return (size_t)(2 * L + W + (random_order ? L + L / 4 : W) + q * L) * 4;
}

// a5, field variant: the columns of the old and the new colour after an accepted change at site fs,
//   ha[j] -= Jq[|j0 + j - fs|],  hb[j] += Jq[|j0 + j - fs|]   for the n sites j0 .. j0 + n - 1 held in ha, hb
// (distances folded to <= L/2 when FOLD: J then only needs the entries 0..L/2).  Each thread takes the sites
// tid, tid + T, ..: four at a time, all twelve loads issued before the eight stores (the three arrays do not
// overlap, a != b; written this way because the compiler must assume that they do and would serialise them).
template <bool FOLD>
__device__ __forceinline__ void field_column_update(int32_t* ha, int32_t* hb, const int32_t* J, int n, int j0, int fs,
                                                    int L, int tid) {
    constexpr int T = FIELD_THREADS;
    if (n < 4 * T) {   // short columns: one site at a time
        for (int j = tid; j < n; j += T) {
            int dist = j0 + j - fs;
            dist = dist < 0 ? -dist : dist;
            if (FOLD) dist = dist > (L >> 1) ? L - dist : dist;
            const int32_t Jv = J[dist];
            ha[j] -= Jv;
            hb[j] += Jv;
        }
        return;
    }
    for (int jb = tid; jb < n; jb += 4 * T) {
        int32_t jv[4], av[4], bv[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const int j = jb + u * T;
            if (j < n) {
                int dist = j0 + j - fs;
                dist = dist < 0 ? -dist : dist;
                if (FOLD) dist = dist > (L >> 1) ? L - dist : dist;
                jv[u] = J[dist];   // J[0] = 0: the site's own field is unchanged
                av[u] = ha[j];
                bv[u] = hb[j];
            }
        }
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const int j = jb + u * T;
            if (j < n) {
                ha[j] = av[u] - jv[u];
                hb[j] = bv[u] + jv[u];
            }
        }
    }
}

template <bool RANDOM, int BITS>
__global__ void __launch_bounds__(FIELD_THREADS, 1)
sweep_field_kernel(Dev d, long long sweep0, int n_sweeps, int do_swap) {
    extern __shared__ uint32_t smem_f[];
    const int L = d.L, W = d.W, q = d.q;
    int32_t* J = (int32_t*)smem_f;
    int32_t* theta = J + L;
    uint32_t* sp = (uint32_t*)(theta + L);
    uint32_t* bq = sp + W;                                  // sequential order: proposed colours, packed
    int32_t* site = (int32_t*)(sp + W);                     // RANDOM: site of step n ...
    uint8_t* kk = (uint8_t*)(site + L);                     // ... and its draw k in 0..q-2
    int32_t* h = RANDOM ? (int32_t*)(kk + L) : (int32_t*)(bq + W);
    __shared__ int s_flip[5];
    __shared__ int s_cnt[PT_QMAX];
    constexpr int PER = 32 / BITS;
    constexpr uint32_t CMASK = (1u << BITS) - 1u;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int e = blockIdx.x / d.n_rep, t = blockIdx.x % d.n_rep;
    const int st = d.perm[blockIdx.x];
    const size_t x = (size_t)e * d.n_rep + st;
    uint32_t* g_sp = d.spins + x * W;
    int32_t* g_h = d.h + x * (size_t)q * L;

    for (int r = tid; r < L; r += FIELD_THREADS) J[r] = d.Jq[r];
    for (int w = tid; w < W; w += FIELD_THREADS) sp[w] = g_sp[w];
    for (int k = tid; k < q * L; k += FIELD_THREADS) h[k] = g_h[k];
    long long E = d.E[x];
    const double scale = d.thr_scale[t];
    const uint32_t c3 = ((uint32_t)(d.ens_base + e) << 4) | TAG_SWEEP;
    ObsAcc oa;
    __syncthreads();

    for (int s = 0; s < n_sweeps; ++s) {
        const uint32_t sweep = (uint32_t)(sweep0 + s + 1);
        if (RANDOM) {
            for (int n = tid; n < L; n += FIELD_THREADS) {
                const Philox4 p = philox4x32_10((uint32_t)n, sweep, (uint32_t)t, c3, d.key0, d.key1);
                site[n] = (int32_t)__umulhi(p.w3, (uint32_t)L);
                kk[n] = (uint8_t)__umulhi(p.w0, (uint32_t)(q - 1));
                theta[n] = accept_threshold(uniform53(p.w1, p.w2), scale);
            }
        }
        // proposals and thresholds of all sites (A6, A7, A9), one word of PER sites per thread
        for (int w = tid; !RANDOM && w < W; w += FIELD_THREADS) {
            const uint32_t word = sp[w];
            uint32_t bword = 0;
#pragma unroll
            for (int n = 0; n < PER; ++n) {
                const int i = PER * w + n;
                const Philox4 p = philox4x32_10((uint32_t)i, sweep, (uint32_t)t, c3, d.key0, d.key1);
                const uint32_t a = (word >> (BITS * n)) & CMASK;
                const uint32_t k = __umulhi(p.w0, (uint32_t)(q - 1));
                const uint32_t b = k + (k >= a ? 1u : 0u);
                bword |= b << (BITS * n);
                theta[i] = accept_threshold(uniform53(p.w1, p.w2), scale);
            }
            bq[w] = bword;
        }
        __syncthreads();

        int pos = 0;
        while (true) {
            if (warp == 0) {
                int f = L, fi = 0, fa = 0, fb = 0, fdE = 0;
                for (int base = pos; base < L; base += 32) {
                    const int n = base + lane;     // step; sequential order: step n visits site n
                    int i = n, a = 0, b = 0, dE = 0;
                    bool acc = false;
                    if (n < L) {
                        if (RANDOM) i = site[n];
                        a = get_colour(sp, i, BITS);
                        if (RANDOM) { const int k = kk[n]; b = k + (k >= a ? 1 : 0); }
                        else b = get_colour(bq, i, BITS);
                        dE = h[a * L + i] - h[b * L + i];
                        acc = dE <= theta[n];
                    }
                    const unsigned m = __ballot_sync(0xffffffffu, acc);
                    if (m) {
                        const int src = __ffs(m) - 1;
                        f = base + src;
                        fi = __shfl_sync(0xffffffffu, i, src);
                        fa = __shfl_sync(0xffffffffu, a, src);
                        fb = __shfl_sync(0xffffffffu, b, src);
                        fdE = __shfl_sync(0xffffffffu, dE, src);
                        break;
                    }
                }
                if (lane == 0) { s_flip[0] = f; s_flip[1] = fa; s_flip[2] = fb; s_flip[3] = fdE; s_flip[4] = fi; }
            }
            __syncthreads();
            const int f = s_flip[0];
            if (f >= L) break;
            const int a = s_flip[1], b = s_flip[2], fs = s_flip[4];   // fs: the site of step f
            field_column_update<false>(h + a * L, h + b * L, J, L, 0, fs, L, tid);
            if (tid == 0) {
                const int sh = (fs % PER) * BITS;
                sp[fs / PER] = (sp[fs / PER] & ~(CMASK << sh)) | ((uint32_t)b << sh);
                E += s_flip[3];
                oa.acc += 1;
            }
            pos = f + 1;
            __syncthreads();
        }
        // a8: sample after the sweep, before the swap event (A15)
        const int nmax = count_nmax(sp, W, q, BITS, s_cnt);
        if (tid == 0) { oa.att += L; oa.sample(E, nmax); }
        __syncthreads();
    }

    for (int w = tid; w < W; w += FIELD_THREADS) g_sp[w] = sp[w];
    for (int k = tid; k < q * L; k += FIELD_THREADS) g_h[k] = h[k];
    if (tid == 0) { d.E[x] = E; oa.flush(d.obs + blockIdx.x); }
    if (do_swap) arrive_and_swap(d, e, (uint32_t)(sweep0 + n_sweeps));
}


// ---------------------------------------------------------------------------
// Local-field variant beyond one SM's shared memory (north_star (3): "one CTA or
// thread-block cluster per replica ... (or DSMEM)"): one thread-block CLUSTER of C = 2, 4 or 8 CTAs per replica.
// CTA c of the cluster owns the sites lo .. lo + L/C - 1, lo = c L/C: their packed spins, proposals, thresholds and
// the columns h[k][i] of the local fields live in ITS shared memory (q L/C words instead of q L); every CTA keeps the
// half coupling table Jq[0..L/2] (Jq[r] = Jq[L-r], A3).  The sweep is the same sequential scan as above: the CTA that
// owns the next site scans its slice for the next accepting site (warp 0, 32 sites at a time) and writes ONE record
// -- next position, site, colours a -> b, dE -- into the shared memory of EVERY CTA of the cluster through DSMEM
// (mapa + st.shared::cluster); after a cluster barrier (release/acquire) every CTA applies the change to its own
// columns, h[a][j] -= Jq[|j-f|], h[b][j] += Jq[|j-f|] for its L/C sites j, so a column update takes 1/C of the time
// it takes a single CTA.  A record without a site hands the scan to the next CTA at the end of a slice.  Records are
// double buffered by step parity: record n+2 is written only after every CTA has arrived at barrier n+1, i.e. after
// it has read record n.  All CTAs see all records, so each keeps the running energy; CTA 0 owns the observables and
// gets the colour counts of the other slices through DSMEM.  Sequential site order only (A5).
// dynamic smem (32-bit words): J[L/2 + 8] | theta[L/C] | sp[W/C] | bq[W/C] | h[q L/C]
// ---------------------------------------------------------------------------
constexpr int FIELD_CLUSTER_MAX = 8;   // portable cluster size

__host__ __device__ inline size_t field_cluster_smem_bytes(int L, int q, int C) {
    const int Ls = L / C, Ws = q <= 16 ? Ls / 8 : Ls / 4;
    return (size_t)((L / 2 + 8) + Ls + 2 * Ws + q * Ls) * 4;
}
// every slice is a whole number of packed words
__host__ __device__ inline bool field_cluster_divides(int L, int C) { return (L % (8 * C)) == 0; }

__device__ __forceinline__ unsigned cluster_ctarank() {
    unsigned r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
    return r;
}
__device__ __forceinline__ unsigned cluster_nctarank() {
    unsigned r;
    asm volatile("mov.u32 %0, %%cluster_nctarank;" : "=r"(r));
    return r;
}
// all threads of all CTAs of the cluster; the arriving threads' shared-memory writes (local and remote) are visible
// to every thread behind the wait
__device__ __forceinline__ void cluster_sync_all() {
    asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}
// address of the same shared-memory variable in CTA `rank` of the cluster (shared::cluster window)
__device__ __forceinline__ uint32_t cluster_map(const void* p, unsigned rank) {
    uint32_t a = (uint32_t)__cvta_generic_to_shared(p), r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(a), "r"(rank));
    return r;
}
__device__ __forceinline__ void st_cluster_v4(uint32_t addr, int4 v) {
    asm volatile("st.shared::cluster.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(addr), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w)
                 : "memory");
}
__device__ __forceinline__ void st_cluster_b32(uint32_t addr, int v) {
    asm volatile("st.shared::cluster.b32 [%0], %1;" ::"r"(addr), "r"(v) : "memory");
}

template <int BITS>
__global__ void __launch_bounds__(FIELD_THREADS, 1)
sweep_field_cluster_kernel(Dev d, long long sweep0, int n_sweeps, int do_swap) {
    extern __shared__ uint32_t smem_fc[];
    constexpr int PER = 32 / BITS;
    constexpr uint32_t CMASK = (1u << BITS) - 1u;
    const int C = (int)cluster_nctarank(), cr = (int)cluster_ctarank();
    const int L = d.L, q = d.q, H = L / 2;
    const int Ls = L / C, Ws = Ls / PER, lo = cr * Ls;
    int32_t* J = (int32_t*)smem_fc;
    int32_t* theta = J + (H + 8);
    uint32_t* sp = (uint32_t*)(theta + Ls);
    uint32_t* bq = sp + Ws;
    int32_t* h = (int32_t*)(bq + Ws);
    __shared__ __align__(16) int s_rec[2][4];                    // the step's record, written by the scanning CTA
    __shared__ int s_cnt[PT_QMAX];
    __shared__ int s_call[FIELD_CLUSTER_MAX][PT_QMAX];           // CTA 0: colour counts of every slice

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int rep = blockIdx.x / C;                              // clusters are C consecutive CTAs of the grid
    const int e = rep / d.n_rep, t = rep % d.n_rep;
    const int st = d.perm[rep];
    const size_t x = (size_t)e * d.n_rep + st;
    uint32_t* g_sp = d.spins + x * d.W + lo / PER;
    int32_t* g_h = d.h + x * (size_t)q * L + lo;

    for (int r = tid; r <= H; r += FIELD_THREADS) J[r] = d.Jq[r];
    for (int w = tid; w < Ws; w += FIELD_THREADS) sp[w] = g_sp[w];
    for (int k = 0; k < q; ++k)
        for (int jj = tid; jj < Ls; jj += FIELD_THREADS) h[k * Ls + jj] = g_h[(size_t)k * L + jj];
    long long E = d.E[x];
    const double scale = d.thr_scale[t];
    const uint32_t c3 = ((uint32_t)(d.ens_base + e) << 4) | TAG_SWEEP;
    ObsAcc oa;
    __syncthreads();
    cluster_sync_all();   // every CTA of the cluster is running: its shared memory may be written from now on
    int par = 0;

    for (int s = 0; s < n_sweeps; ++s) {
        const uint32_t sweep = (uint32_t)(sweep0 + s + 1);
        // proposals and thresholds of the own sites (A6, A7, A9)
        for (int w = tid; w < Ws; w += FIELD_THREADS) {
            const uint32_t word = sp[w];
            uint32_t bword = 0;
#pragma unroll
            for (int n = 0; n < PER; ++n) {
                const int ii = PER * w + n;
                const Philox4 p = philox4x32_10((uint32_t)(lo + ii), sweep, (uint32_t)t, c3, d.key0, d.key1);
                const uint32_t a = (word >> (BITS * n)) & CMASK;
                const uint32_t k = __umulhi(p.w0, (uint32_t)(q - 1));
                const uint32_t b = k + (k >= a ? 1u : 0u);
                bword |= b << (BITS * n);
                theta[ii] = accept_threshold(uniform53(p.w1, p.w2), scale);
            }
            bq[w] = bword;
        }
        __syncthreads();

        int pos = 0;   // next site of the sweep (global index): the same in every CTA of the cluster
        while (pos < L) {
            if (pos / Ls == cr && warp == 0) {
                int nxt = lo + Ls, fs = -1, fab = 0, fdE = 0;   // no site found: the scan moves on to the next slice
                for (int base = pos - lo; base < Ls; base += 32) {
                    const int n = base + lane;
                    int a = 0, b = 0, dE = 0;
                    bool acc = false;
                    if (n < Ls) {
                        a = get_colour(sp, n, BITS);
                        b = get_colour(bq, n, BITS);
                        dE = h[a * Ls + n] - h[b * Ls + n];
                        acc = dE <= theta[n];
                    }
                    const unsigned m = __ballot_sync(0xffffffffu, acc);
                    if (m) {
                        const int src = __ffs(m) - 1;
                        fs = lo + base + src;
                        nxt = fs + 1;
                        fab = __shfl_sync(0xffffffffu, a | (b << 8), src);
                        fdE = __shfl_sync(0xffffffffu, dE, src);
                        break;
                    }
                }
                if (lane < C) st_cluster_v4(cluster_map(&s_rec[par][0], (unsigned)lane), make_int4(nxt, fs, fab, fdE));
                __syncwarp();
            }
            cluster_sync_all();
            const int4 rec = *reinterpret_cast<const int4*>(&s_rec[par][0]);
            par ^= 1;
            const int fs = rec.y;
            if (fs >= 0) {
                const int a = rec.z & 255, b = rec.z >> 8;
                field_column_update<true>(h + a * Ls, h + b * Ls, J, Ls, lo, fs, L, tid);
                if (tid == 0) {
                    E += rec.w;
                    oa.acc += 1;
                    if (fs >= lo && fs < lo + Ls) {
                        const int ii = fs - lo, sh = (ii % PER) * BITS;
                        sp[ii / PER] = (sp[ii / PER] & ~(CMASK << sh)) | ((uint32_t)b << sh);
                    }
                }
            }
            pos = rec.x;
            __syncthreads();
        }
        // a8: sample after the sweep, before the swap event (A15); the colour counts of the slices meet in CTA 0
        count_nmax(sp, Ws, q, BITS, s_cnt);
        if (tid < q) st_cluster_b32(cluster_map(&s_call[cr][tid], 0u), s_cnt[tid]);
        cluster_sync_all();
        if (cr == 0 && tid == 0) {
            int nmax = 0;
            for (int k = 0; k < q; ++k) {
                int c = 0;
                for (int cc = 0; cc < C; ++cc) c += s_call[cc][k];
                nmax = max(nmax, c);
            }
            oa.att += L;
            oa.sample(E, nmax);
        }
        __syncthreads();
    }

    for (int w = tid; w < Ws; w += FIELD_THREADS) g_sp[w] = sp[w];
    for (int k = 0; k < q; ++k)
        for (int jj = tid; jj < Ls; jj += FIELD_THREADS) g_h[(size_t)k * L + jj] = h[k * Ls + jj];
    if (cr == 0 && tid == 0) { d.E[x] = E; oa.flush(d.obs + rep); }
    cluster_sync_all();   // nobody leaves while its shared memory may still be addressed
    if (do_swap && cr == 0) arrive_and_swap(d, e, (uint32_t)(sweep0 + n_sweeps));
}

}  // namespace ptk

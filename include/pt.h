/* include/pt.h -- C ABI of libpt: the parallel-tempering Metropolis sweep of the
 * one-dimensional q-state Potts model with periodic long-range couplings
 * (arXiv 1308.5426; citations are PAPER.md:<line> plus the equation/section).
 *
 * The model (Eqs. 1-7): spins s_i in {1..q} (Eq. 1) on a ring
 * of L sites, H = -sum_{i<j} J*(|i-j|) delta(s_i,s_j) (Eqs. 2-3, each unordered
 * pair once -- reading A1 of DESIGN.md), J*(r) = sum_n |r+nL|^-(1+sigma)
 * (Eqs. 4-5) evaluated through the Hurwitz-zeta closed form (Eqs. 6-7).
 * The library quantises J* to int32 fixed point at scale 2^24,
 * Jq[r] = round(J*(r) 2^24), so every energy below is an exact integer in
 * units of 2^-24 and independent of summation order.
 *
 * The method (Eqs. 8-9; 110-128, section 4.2): n_rep replicas
 * ("slots", one per inverse temperature) per ensemble; one sweep = L
 * single-spin Metropolis steps (Eq. 8) in site order 0..L-1 on every replica;
 * a swap event = replica exchange (Eq. 9) between neighbouring slots, pairs
 * (t,t+1) with t even first, then t odd.  Randomness is
 * Philox-4x32-10 keyed by (seed; ensemble, slot, sweep, site), so a trajectory
 * is a pure function of the arguments of pt_create and the number of sweeps.
 *
 * Conventions
 *  - All pointers are HOST pointers unless the function name ends in _dev, in
 *    which case they are DEVICE pointers on the context's device.  The caller
 *    owns every in/out array; the library owns all state behind pt_ctx.
 *  - Arrays over replicas are indexed [ensemble][slot], slot = position in
 *    `betas`; "neighbouring temperatures" = adjacent slots.
 *  - Every function returns 0 (PT_OK) or a negative pt_status; the message of
 *    the last failure on the calling thread is returned by pt_last_error().
 *    No C++ exception crosses this boundary.  Calls are synchronous: results
 *    are complete when the call returns (kernels run on the stream given to
 *    pt_set_stream, default stream otherwise).
 *  - A context must not be used from two threads at once.  Every call runs on
 *    the device the context was created on and restores the caller's current
 *    device before it returns.
 */
#ifndef PT_H_
#define PT_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct pt_ctx pt_ctx; /* opaque; created by pt_create, freed by pt_destroy */

typedef enum {
    PT_OK = 0,
    PT_EINVAL = -1,    /* bad argument (see each call) */
    PT_EOVERFLOW = -2, /* sum_r Jq[r] >= 2^31: dE would not fit int32 (sigma too small) */
    PT_ENOMEM = -3,    /* host or device allocation failed */
    PT_ECUDA = -4,     /* CUDA runtime error, no device, or not an sm_100 device */
    PT_ECAPACITY = -5  /* no sweep variant fits the shared memory of one SM (field variant: of a cluster of 8 SMs) for (L,q) */
} pt_status;

/* Sweep variants (pt_set_variant).  Both produce bit-identical trajectories.
 *  PT_VARIANT_FIELD : per-colour local fields h[k][i] = sum_{j!=i} Jq[|i-j|][s_j==k]
 *                     kept in shared memory; a proposal costs O(1), an accepted
 *                     change updates two columns of h (north_star (3)).  Where
 *                     L*q*4 bytes + tables exceed one SM's 227 KB, a replica takes
 *                     a thread-block cluster of 2, 4 or 8 CTAs, each holding the
 *                     fields of L/C consecutive sites (sequential site order only;
 *                     needs L % (8 C) == 0; DSMEM carries one 16-byte record per
 *                     accepted change to every CTA of the cluster).
 *  PT_VARIANT_DIRECT: dE = sum_j Jq[|i-j|]([s_j==a]-[s_j==b]) summed directly
 *                     (PAPER.md:118-124), for blocks of 32 consecutive sites at a
 *                     time, with exact integer corrections for the changes
 *                     accepted inside the block.  Needs L % 64 == 0,
 *                     64 <= L <= 10240 (q > 8: L <= 9664, shared memory) and sum_r Jq[r] < 2^30 - 1.
 *  PT_VARIANT_AUTO  : DIRECT where it applies, else FIELD.
 * Environment: PT_VARIANT=direct|field|auto sets the variant chosen by pt_create; PT_PERSISTENT=0|1|2 the launch
 * policy of the direct variant (0: one launch per swap interval; 1, default: persistent launches with the swap events
 * inside the kernel for contexts that take at least a third of the SMs; 2: whenever all replicas can be co-resident);
 * PT_MINB=1|2|4 forces the 168-, the 80- or (1024 < L <= 2048) the 128-register build of the direct sweep kernel
 * (experiments; default: by size and replica count).  PT_FIELD_CLUSTER=2|4|8 runs the field variant on clusters of
 * that size also where one CTA would hold the replica (tests, measurements).
 * PT_CW=2 (L = 4096, q <= 8): two chain warps instead of four (bit-identical, measured slower: an experiment).
 * PT_FAR=1 (L = 4096, q <= 8) selects the far form of the bulk sum (8-bit coupling residuals beyond 1000 sites;
 * bit-identical results, measured slower than the default form: an experiment kept for reference). */
enum { PT_VARIANT_AUTO = 0, PT_VARIANT_FIELD = 1, PT_VARIANT_DIRECT = 2, PT_VARIANT_FP32 = 3, PT_VARIANT_FP64 = 4 };
/* PT_VARIANT_FP32 / PT_VARIANT_FP64: the paper's own arithmetic as a COMPARISON variant ("single
 * precision ... rounding errors"; :110-124: one thread block per replica, each of its 128 threads sums a subset of the
 * pair terms of dE, then a tree reduction; :216 "double precision ... about half the speed").  Same quantised model
 * (couplings (T)(Jq[r] 2^-24)), same random streams; dE and the running energy in T = float / double, Eqs. 8-9 in
 * fp64 on those values.  fp64 reproduces the integer trajectory exactly; fp32 measures what single precision costs.
 * pt_energy(recompute = 0) returns the running value rounded to fixed point; leaving the variant recounts the
 * energies exactly.  Never chosen by AUTO; swap events by one launch per swap interval. */

/* Cumulative per-slot accumulators since pt_create (the caller differences two
 * snapshots to discard burn-in).  Sampled after every sweep, before the swap
 * event, for the slot the configuration occupied during the sweep
 * ("at the end of the Metropolis cycle we calculate the total
 * energy"; Eq. 10 PAPER.md:136-140 for the magnetisation).
 * E is the TOTAL energy in fixed point (units 2^-24).  Nmax = max_k N_k, so
 * that M = (q Nmax/L - 1)/(q-1) (Eq. 10). */
typedef struct {
    int64_t n_samples;
    int64_t sum_E;
    uint64_t sum_E2_lo; /* sum of E^2 as a 128-bit integer: low 64 bits ... */
    int64_t sum_E2_hi;  /* ... high 64 bits */
    int64_t sum_Nmax;
    int64_t sum_Nmax2;
    int64_t flip_attempts; /* Metropolis steps, Eq. 8 */
    int64_t flip_accepts;
    int64_t swap_attempts; /* Eq. 9, pair (t,t+1) recorded at slot t */
    int64_t swap_accepts;
    int64_t near_ties;     /* -1: not counted by this library (the CPU oracle counts them) */
    /* Higher moments for the cumulants U_E = <E^4>/<E^2>^2 (Eq. 11) and
     * V_M = 1 - <M^4>/(3<M^2>^2) (Eq. 12); M^4 is a polynomial of degree 4 in Nmax (Eq. 10).
     * Valid while Nmax^3 sums fit int64 (L <= 2^14 for any realistic number of samples). */
    uint64_t sum_E4[4];    /* sum of E^4 as a 256-bit unsigned integer, little-endian 64-bit limbs */
    int64_t sum_Nmax3;
    uint64_t sum_Nmax4_lo; /* sum of Nmax^4 as a 128-bit integer: low 64 bits ... */
    int64_t sum_Nmax4_hi;  /* ... high 64 bits */
} pt_obs;

/* Create a context on the current CUDA device: evaluates J* (Eqs. 5-7) on the
 * device in fp64 and quantises it, draws the hot start (spins uniform in
 * {1..q} from the Philox stream) and computes every replica's total energy.
 *  L      : ring length, L >= 8 and L % 8 == 0 (8 spins per 32-bit word)
 *  q      : number of colours, 2 <= q <= 64.  q <= 16: 4 bits per spin, every variant.  16 < q <= 64: 8 bits per
 *           spin (4 spins per word); the field and the floating-point variants only (the direct kernels are built
 *           on nibble tables), so PT_VARIANT_AUTO resolves to PT_VARIANT_FIELD and needs L*q*4 bytes + tables of
 *           shared memory, of one SM or spread over a cluster of up to 8 (PT_ECAPACITY beyond that)
 *  sigma  : decay exponent of Eq. 4, finite and > 0
 *  n_ens  : independent ensembles (same model, different random streams) >= 1
 *  n_rep  : replicas per ensemble >= 1
 *  betas  : [n_rep] inverse temperatures (k_B = 1), finite, >= 0,
 *           any order; shared by all ensembles
 *  seed   : Philox key
 * Errors: PT_EINVAL, PT_EOVERFLOW, PT_ENOMEM, PT_ECUDA, PT_ECAPACITY. *out is
 * set to NULL on failure. */
int pt_create(pt_ctx** out, int L, int q, double sigma, int n_ens, int n_rep,
              const double* betas, uint64_t seed);

/* As pt_create, with the ensemble index of this context's first ensemble set
 * to ens_base (0 <= ens_base, ens_base + n_ens <= 2^28): ensemble e of this
 * context draws the random stream of global ensemble ens_base + e.  This is how
 * ensembles are sharded over processes / GPUs without any communication. */
int pt_create_ex(pt_ctx** out, int L, int q, double sigma, int n_ens, int n_rep,
                 const double* betas, uint64_t seed, int ens_base);

/* Slot-sharded context: ONE ensemble of n_rep replicas spread over several processes / GPUs.
 * Every process creates the context with the same arguments except (rep_base, n_local): it sweeps the n_local
 * configurations with storage index rep_base .. rep_base + n_local - 1 (at creation storage index = slot), and keeps
 * a full copy of the slot -> storage permutation.  Configurations never leave their process; at a swap event
 * (Eq. 9) only energies are exchanged: every process passes the energies of ALL configurations, in
 * storage order (an all-gather of pt_energy_storage_dev), to pt_swap_external, which takes the same decisions
 * everywhere from the slot-keyed random stream and moves the temperature labels.  pt_sweeps must be called with
 * swap_every = 0.  The accumulators of a slot are gathered by whichever process holds its configuration: the
 * ensemble's observables are the field-wise sums over the processes (swap counters: process with rep_base = 0).
 * Needs the direct variant (PT_EINVAL otherwise), 0 <= rep_base, n_local >= 1, rep_base + n_local <= n_rep. */
int pt_create_shard(pt_ctx** out, int L, int q, double sigma, int n_rep, const double* betas, uint64_t seed,
                    int ens_base, int rep_base, int n_local);

/* Slot-sharded contexts: running energies of the local configurations, E_out_dev[n_local] (DEVICE pointer),
 * storage order. */
int pt_energy_storage_dev(pt_ctx* ctx, int64_t* E_out_dev);

/* Slot-sharded contexts: one swap event (even pairs, then odd pairs) after the current sweep, from the energies of
 * all n_rep configurations in storage order, E_all_dev[n_rep] (DEVICE pointer). */
int pt_swap_external(pt_ctx* ctx, const int64_t* E_all_dev);

/* Asynchronous forms of the two calls above: enqueued on the context's stream, no synchronisation (the caller orders
 * its own collective on the same stream and calls pt_sync at the end): one swap event then costs no host round trip. */
int pt_energy_storage_dev_async(pt_ctx* ctx, int64_t* E_out_dev);
int pt_swap_external_async(pt_ctx* ctx, const int64_t* E_all_dev);

/* perm[n_ens*n_rep]: storage index (inside the ensemble) of the configuration at each slot. */
int pt_get_perm(pt_ctx* ctx, int32_t* perm);

void pt_destroy(pt_ctx* ctx); /* NULL is allowed */

/* Advance every replica by n >= 0 sweeps.  With swap_every > 0 a swap event
 * follows each sweep whose global index (counted from pt_create, first sweep
 * = 1) is a multiple of swap_every, so splitting n over several calls changes
 * nothing.  swap_every = 0: never swap.  Errors: PT_EINVAL (n < 0,
 * swap_every < 0), PT_EOVERFLOW (the sweep counter would pass 2^32 - 1: the
 * sweep index is one 32-bit word of the Philox counter), PT_ECUDA. */
int pt_sweeps(pt_ctx* ctx, int64_t n, int swap_every);

/* Total energies E_out[n_ens*n_rep] (fixed point 2^-24).  recompute = 0 returns
 * the running value (E0 + sum of accepted dE); recompute = 1 recounts
 * E = -sum_{i<j} Jq[j-i] [s_i==s_j] from the spins (O(L^2)) and
 * leaves the running value untouched. */
int pt_energy(pt_ctx* ctx, int64_t* E_out, int recompute);
int pt_energy_dev(pt_ctx* ctx, int64_t* E_out_dev, int recompute);

/* out[n_ens*n_rep] accumulators, see pt_obs. */
int pt_observables(pt_ctx* ctx, pt_obs* out);

/* out[n_ens*n_rep*L] colours 1..q (Eq. 1), one byte per spin. */
int pt_get_spins(pt_ctx* ctx, uint8_t* out);
int pt_get_spins_dev(pt_ctx* ctx, uint8_t* out_dev);

/* Replace all configurations (cold starts, resume); recomputes the energies
 * (and local fields).  PT_EINVAL if a colour is outside 1..q (state unchanged).
 * The sweep counter and the accumulators are kept. */
int pt_set_spins(pt_ctx* ctx, const uint8_t* in);

/* Checkpoint / resume.  The state of a context is: the configurations, their running energies,
 * the accumulators and the sweep counter -- the generator is counter based and has no state, and the slot -> storage
 * permutation is not observable.  pt_get_state writes them to host arrays (spins[n_ens*n_rep*L] colours 1..q,
 * E[n_ens*n_rep], obs[n_ens*n_rep], all in slot order).  pt_set_state loads them into a context created with the same
 * arguments: "destroy, create, pt_set_state, continue" is bit-identical to the uninterrupted run.  E may be NULL (the
 * energies are recounted from the spins, O(L^2)); obs may be NULL (the accumulators are kept).  PT_EINVAL: a colour
 * outside 1..q (state unchanged), sweep outside 0 .. 2^32 - 1, or a slot-sharded context. */
int pt_get_state(pt_ctx* ctx, uint8_t* spins, int64_t* E, pt_obs* obs, int64_t* sweep);
int pt_set_state(pt_ctx* ctx, const uint8_t* spins, const int64_t* E, const pt_obs* obs, int64_t sweep);

/* Jq[L]: Jq[0] = 0, Jq[r] = Jq[L-r] = round(J*(r) 2^24). */
int pt_get_couplings(pt_ctx* ctx, int32_t* Jq);

/* Number of sweeps done since pt_create. */
int64_t pt_sweep_counter(pt_ctx* ctx);

/* variant: PT_VARIANT_*.  PT_EINVAL if the variant cannot run this (L,q);
 * PT_ECAPACITY if it does not fit in shared memory.  Switching rebuilds
 * whatever the new variant needs from the spins; the trajectory is unchanged. */
int pt_set_variant(pt_ctx* ctx, int variant);
int pt_get_variant(pt_ctx* ctx); /* the variant that pt_sweeps runs (FIELD or DIRECT) */

/* The launch plan of the context as one line of text (what pt_sweeps would launch now), e.g.
 *   "direct: threads=384 regs=155 resident_ctas=148 near_window=96 near_quads=1 chain_warps=4 persistent=1"
 *   "field: cluster=4 threads=512 smem=186400"
 * out: caller's buffer of n bytes (host), NUL-terminated on return; a longer line is truncated.  Returns PT_OK,
 * PT_EINVAL (NULL arguments, n < 1) or PT_ECUDA.  For logs, bench lines and tests of the launch policy
 * (DESIGN.md sections 6.1b, 6.2); nothing of the path depends on it. */
int pt_describe(pt_ctx* ctx, char* out, int n);

/* Site order of a sweep (reading A5 of DESIGN.md).  PT_ORDER_SEQUENTIAL (default, BASELINE configs): sites 0..L-1
 * in order.  PT_ORDER_RANDOM ("L Metropolis steps ... an average of one Monte Carlo step per
 * spin"): step n = 0..L-1 of a sweep visits site mulhi32(w3, L) of the Philox draw keyed by (n, sweep, slot), which
 * also gives the proposal and the uniform of the step.  Random order runs in the field variant (it is selected by
 * this call; PT_ECAPACITY if the local-field table and the step lists do not fit in shared memory; pt_set_variant
 * to another variant is refused while it is on).  Errors: PT_EINVAL, PT_ECAPACITY. */
enum { PT_ORDER_SEQUENTIAL = 0, PT_ORDER_RANDOM = 1 };
int pt_set_site_order(pt_ctx* ctx, int order);

/* Kernels are launched on `cuda_stream` (a cudaStream_t; NULL = default stream). */
int pt_set_stream(pt_ctx* ctx, void* cuda_stream);

/* Asynchronous form of pt_sweeps for timing with CUDA events: enqueues the
 * launches on the context's stream and returns without synchronising.
 * *n_launches (may be NULL) receives the number of kernels enqueued. */
int pt_sweeps_async(pt_ctx* ctx, int64_t n, int swap_every, int64_t* n_launches);

/* Blocks until the context's stream is idle; returns PT_ECUDA if a kernel failed, or if a swap barrier inside a
 * persistent launch timed out (30 s of wall-clock time without the arrival of a co-resident CTA: the state of the
 * context is lost). */
int pt_sync(pt_ctx* ctx);

/* Instruction-rate micro-benchmarks on the current device (the ALU roofline of the direct sweep kernel
 * rests on the measured issue rate of IDP.2A, not on a datasheet).  rates[p*4 + (w-1)] = lane-operations per clock
 * and SM of pattern p with w = 1..4 warps per SM sub-partition, timed with clock64() inside the kernel (median over
 * the SMs).  Patterns: 0 IDP.2A, 1 IDP.4A, 2 IMAD, 3 PRMT, 4 LOP3, 5 the bulk loop's mix of 1 PRMT + 2 IDP.2A
 * (counting the IDP.2A only), 6 1 LOP3 + 2 IDP.2A (ditto), 7 LDS.128 in bytes per clock and SM, 8 1 PRMT + 4 IDP.2A,
 * 9 the mirror-paired mix 2 PRMT + 1 ADD + 2 IDP.2A (IDP.2A counted; 4 pair terms per IDP.2A lane-operation),
 * 10 the bulk tile of the direct sweep kernel as it stands (8 sites x 16 steps: one PRMT on the site's two table
 * registers and two IDP.2A on 39 packed coupling registers per step and site; IDP.2A counted), 11 the same tile in the
 * far form of PT_FAR (one PRMT and one IDP.4A per step and site; the IDP.4A counted, each standing for two IDP.2A).
 * One IDP.2A lane-operation is two multiply-accumulates (one per pair term of the energy sum).
 * n = number of doubles `rates` holds, >= 4 * PT_PEAK_PATTERNS.  Errors: PT_EINVAL, PT_ENOMEM, PT_ECUDA. */
#define PT_PEAK_PATTERNS 12
int pt_measure_peaks(double* rates, int n);

/* Total energies of caller-supplied configurations WITHOUT ANY ALLOCATION (for callers that cannot call cudaMalloc:
 * code under CUDA graph capture, tight serving loops, harnesses that forbid it).  The same O(L^2) recount as
 * pt_energy(recompute = 1) -- Eq. 2 in reading A1 with each unordered pair once, "the total energy of
 * each replica", on the quantised couplings Jq[r] = round(J*(r) 2^24) of Eqs. 5-7 (A16) -- but on the current device,
 * without a context: the coupling table and the packed spins it needs live in a file-scope device array of
 * 64 + PT_STATIC_MAX_L + PT_STATIC_MAX_SITES/4 32-bit words (1 114 368 bytes) that every GPU loading the library holds
 * until exit.  No cudaMalloc, cudaFree or allocating library routine is called.
 *  L, q, sigma : the model, as for pt_create; L % 8 == 0, 8 <= L <= PT_STATIC_MAX_L, 2 <= q <= 64
 *  spins_dev   : DEVICE pointer, [n_conf][L] bytes, API colours 1..q (A4); not modified; owned by the caller
 *  n_conf      : configurations, >= 1, n_conf * L <= PT_STATIC_MAX_SITES
 *  E_out_dev   : DEVICE pointer, [n_conf] int64, receives E in fixed point 2^-24; owned by the caller
 *  status_dev  : DEVICE pointer to one int or NULL: receives 0, or 1 if some colour was outside 1..q (the energies
 *                of that call are then meaningless)
 *  cuda_stream : a cudaStream_t (NULL = default stream).  The call only ENQUEUES (one memset + 3-4 kernels) and
 *                returns; outputs are complete when that stream work is.
 * All calls share the one scratch array, which keeps the last call's contents (every call clears or overwrites what
 * it reads): calls that OVERLAP on the GPU -- different streams without an ordering between them, or two host
 * threads on one device -- race.  Calls on one stream, or ordered by events, are safe.
 * Errors: PT_EINVAL (arguments), PT_ECAPACITY (L or n_conf * L beyond the maxima: split the call), PT_ECUDA. */
#define PT_STATIC_MAX_L 16384
#define PT_STATIC_MAX_SITES 1048576
int pt_energy_static(int L, int q, double sigma, const uint8_t* spins_dev, int n_conf, int64_t* E_out_dev,
                     int* status_dev, void* cuda_stream);

const char* pt_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* PT_H_ */

// oracle/pt_oracle.cpp -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// A plain, slow, obviously-correct CPU restatement of the hot path of
// "GPU-based simulation of the long-range Potts model via parallel tempering"
// (arXiv 1308.5426; PAPER.md).  It follows the paper step by step in the
// paper's order and notation, in the readings A1-A16 of SURVEY.md 8(c) that
// DESIGN.md restates.  Only tests/, __graft_entry__.smoke() and bench.py's
// cpu_baseline / --impl reference legs may build, load or call this file.
// It shares no code, header, table or constant generator with the CUDA path
// (paper_1308_5426_b200/csrc); neither side includes the other.
//
// Parity pins (tests/test_oracle_*.py, all `-m "not gpu"`):
//   orc_jstar / orc_couplings : Eq. 5 brute-force image sum, sigma=1 closed
//       form (pi/L)^2/sin^2(pi r/L), sum rule 2 zeta(1+sigma)(1-L^-(1+sigma)),
//       mpmath/scipy Hurwitz zeta, symmetry J*(r)=J*(L-r)
//   orc_philox                : Random123 known-answer vectors
//   orc_delta_e / orc_energy  : dE == E(after)-E(before) by O(L^2) recount;
//       all-equal ground state; q=2 <-> long-range Ising identity
//   orc_sweeps                : exact Boltzmann enumeration L=8,q=3 (6561
//       states) within 3 sigma, with and without swaps; beta=0 <delta>=1/q;
//       field mode == direct mode bit for bit; call-splitting invariance;
//       threaded == single-threaded
//   orc_sweeps_arith (the paper's floating-point arithmetic as a comparison mode):
//       fp64 mode reproduces the integer trajectory bit for bit (the couplings Jq 2^-24 have 25 significant
//       bits, so every fp64 sum is exact); fp32 mode: dE within the summation error bound of the exact
//       integer value, <E> of the L=8 enumeration within 3 sigma
//   the paper's fp32 error figures and its speedups:
//       PARITY UNPINNED (context only; the fp32 mode MEASURES the rounding error of this build's model)
//
// Arithmetic: couplings evaluated in long double, quantised to int32 at scale
// 2^24 (A16); every dE and E is an exact integer; acceptance in fp64.

#include <cmath>
#include <cstdint>
#include <cstdlib>
#include <cstring>
#include <thread>
#include <vector>

namespace {

// ---------------------------------------------------------------------------
// Eq. 7: Hurwitz zeta  zeta(s,alpha) = sum_{k>=0} (k+alpha)^-s
// evaluated as: first N terms as written, remainder by the Euler-Maclaurin
// formula (integral + half term + Bernoulli corrections).
// ---------------------------------------------------------------------------
long double hurwitz_zeta(long double s, long double alpha) {
    const int N = 24;
    long double sum = 0.0L;
    for (int k = 0; k < N; ++k) sum += powl((long double)k + alpha, -s);
    const long double x = (long double)N + alpha;
    sum += powl(x, 1.0L - s) / (s - 1.0L);   // integral_N^inf (t+alpha)^-s dt
    sum += 0.5L * powl(x, -s);               // half of the first omitted term
    // B_{2m}/(2m)!  for m = 1..7
    static const long double c[7] = {
        1.0L / 12.0L, -1.0L / 720.0L, 1.0L / 30240.0L, -1.0L / 1209600.0L,
        1.0L / 47900160.0L, -691.0L / 1307674368000.0L, 1.0L / 74724249600.0L};
    long double rising = s;                  // s (s+1) ... (s+2m-2)
    long double xp = powl(x, -s - 1.0L);     // x^(-s-2m+1)
    for (int m = 1; m <= 7; ++m) {
        sum += c[m - 1] * rising * xp;
        rising *= (s + (long double)(2 * m - 1)) * (s + (long double)(2 * m));
        xp /= x * x;
    }
    return sum;
}

// Eq. 6: J*(r) = r^-s + L^-s [zeta(s,1+r/L) + zeta(s,1-r/L)],
// s = 1+sigma, valid for 0 < r < L.
long double jstar(int L, long double sigma, int r) {
    const long double s = 1.0L + sigma;
    const long double x = (long double)r / (long double)L;
    return powl((long double)r, -s) +
           powl((long double)L, -s) * (hurwitz_zeta(s, 1.0L + x) + hurwitz_zeta(s, 1.0L - x));
}

// A16/A3: Jq[r] = round(J*(r) 2^24) for 1 <= r <= L/2, mirrored so that the
// integer table is exactly symmetric; Jq[0] = 0 (A2).
void couplings(int L, double sigma, std::vector<int32_t>& Jq) {
    Jq.assign(L, 0);
    for (int r = 1; r <= L / 2; ++r) {
        long long v = llrintl(ldexpl(jstar(L, (long double)sigma, r), 24));
        Jq[r] = (int32_t)v;
        Jq[L - r] = (int32_t)v;
    }
}

// ---------------------------------------------------------------------------
// Philox-4x32-10 (Salmon et al., SC'11), the counter-based generator the
// north_star prescribes; restated from the published algorithm.
// ---------------------------------------------------------------------------
void philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        const uint64_t p0 = (uint64_t)0xD2511F53u * c0;
        const uint64_t p1 = (uint64_t)0xCD9E8D57u * c2;
        const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
        const uint32_t n1 = (uint32_t)p1;
        const uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
        const uint32_t n3 = (uint32_t)p0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// U(w1,w2) in [0,1) with 53 bits (SURVEY 8c RNG).
double uniform53(uint32_t w1, uint32_t w2) {
    const uint64_t m = ((uint64_t)(w1 >> 5) << 26) | (uint64_t)(w2 >> 6);
    return (double)m * (1.0 / 9007199254740992.0);
}

uint32_t mulhi32(uint32_t a, uint32_t b) { return (uint32_t)(((uint64_t)a * b) >> 32); }

enum { TAG_INIT = 0, TAG_SWEEP = 1, TAG_SWAP = 2 };

struct Obs {              // same field order as include/pt.h's pt_obs (declared separately)
    int64_t n_samples, sum_E;
    uint64_t sum_E2_lo; int64_t sum_E2_hi;
    int64_t sum_Nmax, sum_Nmax2;
    int64_t flip_attempts, flip_accepts;
    int64_t swap_attempts, swap_accepts;
    int64_t near_ties;
    // higher moments for the cumulants of Eqs. 11-12
    uint64_t sum_E4[4];                          // sum of E^4 as a 256-bit integer, little-endian 64-bit limbs
    int64_t sum_Nmax3;
    uint64_t sum_Nmax4_lo; int64_t sum_Nmax4_hi; // sum of Nmax^4 as a 128-bit integer
};

struct Replica {
    std::vector<uint8_t> c;     // colours 0..q-1 (A4)
    int64_t E = 0;              // total energy, fixed point 2^24 (A13)
    double Ef = 0.0;            // floating-point modes: running energy in units of 1 (fp32 mode: a float value)
    std::vector<int64_t> h;     // field mode only: h[i*q+k] = sum_{j!=i} Jq[|i-j|] [c_j==k]
};

struct Ctx {
    int L, q, n_ens, n_rep;
    int ens_base = 0;           // global index of this context's first ensemble (enters the RNG counter only)
    double sigma;
    uint64_t seed;
    uint32_t key[2];
    std::vector<double> beta;
    std::vector<int32_t> Jq;
    std::vector<Replica> rep;   // [ens*n_rep + slot]
    std::vector<Obs> obs;       // [ens*n_rep + slot]
    int64_t sweep = 0;          // global sweep counter (A10)
    int site_order = 0;         // 0: sites 0..L-1 in order (A5); 1: step n visits site mulhi32(w3, L) (A5')
    int float_mode = 0;         // 0: exact integers; 1 / 2: the fp32 / fp64 comparison mode has been entered
};

inline int iabs(int x) { return x < 0 ? -x : x; }

// Eq. 2 in reading A1 (each unordered pair once): E = - sum_{i<j} Jq[j-i] delta(c_i,c_j)
int64_t total_energy(const Ctx& C, const std::vector<uint8_t>& c) {
    int64_t E = 0;
    for (int i = 0; i < C.L; ++i)
        for (int j = i + 1; j < C.L; ++j)
            if (c[i] == c[j]) E -= C.Jq[j - i];
    return E;
}

// PAPER.md:124 "the energies corresponding to the flipped spin before and after":
// dE = E(c_i=b) - E(c_i=a) = sum_{j!=i} Jq[|i-j|] ([c_j==a] - [c_j==b])
int64_t delta_e_direct(const Ctx& C, const std::vector<uint8_t>& c, int i, int a, int b) {
    int64_t dE = 0;
    for (int j = 0; j < C.L; ++j) {
        if (j == i) continue;
        dE += (int64_t)C.Jq[iabs(i - j)] * ((c[j] == a) - (c[j] == b));
    }
    return dE;
}

void build_fields(const Ctx& C, Replica& R) {
    R.h.assign((size_t)C.L * C.q, 0);
    for (int i = 0; i < C.L; ++i)
        for (int j = 0; j < C.L; ++j)
            if (j != i) R.h[(size_t)i * C.q + R.c[j]] += C.Jq[iabs(i - j)];
}

// One "Metropolis cycle" of L steps in sequential site
// order (A5) for the replica in slot t of ensemble e; Eq. 8 acceptance.
void metropolis_cycle(Ctx& C, int e, int t, bool field) {
    Replica& R = C.rep[(size_t)e * C.n_rep + t];
    Obs& O = C.obs[(size_t)e * C.n_rep + t];
    const double beta = C.beta[t];
    const int q = C.q, L = C.L;
    for (int n = 0; n < L; ++n) {                         // step n of the cycle
        const uint32_t ctr[4] = {(uint32_t)n, (uint32_t)C.sweep, (uint32_t)t,
                                 ((uint32_t)(C.ens_base + e) << 4) | TAG_SWEEP};
        uint32_t w[4];
        philox4x32_10(ctr, C.key, w);
        // A5: sequential order visits site n; A5' ("an average of one Monte Carlo step per spin"):
        // a site drawn uniformly from the same Philox word group
        const int i = C.site_order ? (int)mulhi32(w[3], (uint32_t)L) : n;
        const int a = R.c[i];
        const int k = (int)mulhi32(w[0], (uint32_t)(q - 1));
        const int b = k + (k >= a);                       // A6: uniform over the other q-1
        int64_t dE;
        if (field) dE = R.h[(size_t)i * q + a] - R.h[(size_t)i * q + b];
        else       dE = delta_e_direct(C, R.c, i, a, b);
        const double x = -(beta * ldexp((double)dE, -24)); // A8: one rounding
        const double p = (dE <= 0) ? 1.0 : exp(x);         // Eq. 8
        const double u = uniform53(w[1], w[2]);
        if (dE > 0 && fabs(u - p) < 1e-12) O.near_ties++;
        O.flip_attempts++;
        if (dE <= 0 || u < p) {                            // A7: strict
            R.c[i] = (uint8_t)b;
            R.E += dE;
            O.flip_accepts++;
            if (field) {
                for (int j = 0; j < L; ++j) {
                    if (j == i) continue;
                    const int64_t J = C.Jq[iabs(i - j)];
                    R.h[(size_t)j * q + a] -= J;
                    R.h[(size_t)j * q + b] += J;
                }
            }
        }
    }
}

// ---------------------------------------------------------------------------
// The paper's own arithmetic as a comparison mode ("single precision ... rounding errors";
// :118-124 and the caption of Listing 2: "each thread sums a subset of pair terms", then a parallel reduction).
// Reading: couplings Jf[r] = (T)(Jq[r] 2^-24), i.e. the SAME quantised model in type T = float or
// double; dE = sum of the 128 thread-partial sums, thread t adding its terms j = t, t+128, ... in increasing j,
// combined by a binary tree (stride 64, 32, .., 1); the terms are +-Jf or 0, so no product is rounded.  The running
// energy is kept in T; Eq. 8 and Eq. 9 are evaluated in fp64 on the T values (libm's expf is not involved).
// ---------------------------------------------------------------------------
template <typename T>
T delta_e_float(const Ctx& C, const std::vector<T>& Jf, const std::vector<uint8_t>& c, int i, int a, int b) {
    T part[128];
    for (int t = 0; t < 128; ++t) {
        T acc = (T)0;
        for (int j = t; j < C.L; j += 128) {
            if (j == i) continue;
            const T J = Jf[iabs(i - j)];
            if (c[j] == a) acc = acc + J;
            else if (c[j] == b) acc = acc - J;
        }
        part[t] = acc;
    }
    for (int s = 64; s >= 1; s >>= 1)
        for (int t = 0; t < s; ++t) part[t] = part[t] + part[t + s];
    return part[0];
}

template <typename T>
void metropolis_cycle_float(Ctx& C, const std::vector<T>& Jf, int e, int t) {
    Replica& R = C.rep[(size_t)e * C.n_rep + t];
    Obs& O = C.obs[(size_t)e * C.n_rep + t];
    const double beta = C.beta[t];
    const int q = C.q, L = C.L;
    T E = (T)R.Ef;
    for (int i = 0; i < L; ++i) {
        const uint32_t ctr[4] = {(uint32_t)i, (uint32_t)C.sweep, (uint32_t)t,
                                 ((uint32_t)(C.ens_base + e) << 4) | TAG_SWEEP};
        uint32_t w[4];
        philox4x32_10(ctr, C.key, w);
        const int a = R.c[i];
        const int k = (int)mulhi32(w[0], (uint32_t)(q - 1));
        const int b = k + (k >= a);
        const T dE = delta_e_float<T>(C, Jf, R.c, i, a, b);
        const double x = -(beta * (double)dE);
        const double p = (dE <= (T)0) ? 1.0 : exp(x);
        const double u = uniform53(w[1], w[2]);
        if (dE > (T)0 && fabs(u - p) < 1e-12) O.near_ties++;
        O.flip_attempts++;
        if (dE <= (T)0 || u < p) {
            R.c[i] = (uint8_t)b;
            E = E + dE;
            O.flip_accepts++;
        }
    }
    R.Ef = (double)E;
    R.E = llrint(ldexp(R.Ef, 24));   // what the accumulators see: the running value in fixed point
}

void swap_event_float(Ctx& C, int e) {
    for (int stage = 0; stage < 2; ++stage) {
        for (int t = stage; t + 1 < C.n_rep; t += 2) {
            Replica& Ra = C.rep[(size_t)e * C.n_rep + t];
            Replica& Rb = C.rep[(size_t)e * C.n_rep + t + 1];
            Obs& O = C.obs[(size_t)e * C.n_rep + t];
            const double d = (C.beta[t] - C.beta[t + 1]) * (Ra.Ef - Rb.Ef);
            const uint32_t ctr[4] = {(uint32_t)t, (uint32_t)C.sweep, 0u, ((uint32_t)(C.ens_base + e) << 4) | TAG_SWAP};
            uint32_t w[4];
            philox4x32_10(ctr, C.key, w);
            const double u = uniform53(w[1], w[2]);
            O.swap_attempts++;
            if (d < 0 && fabs(u - exp(d)) < 1e-12) O.near_ties++;
            if (d >= 0 || u < exp(d)) {
                std::swap(Ra.c, Rb.c);
                std::swap(Ra.E, Rb.E);
                std::swap(Ra.Ef, Rb.Ef);
                O.swap_accepts++;
            }
        }
    }
}

// A15: sample after the sweep, before swaps.  Eq. 10 needs N_max = max_k N_k.
void measure(Ctx& C, int e, int t) {
    const Replica& R = C.rep[(size_t)e * C.n_rep + t];
    Obs& O = C.obs[(size_t)e * C.n_rep + t];
    std::vector<int64_t> cnt(C.q, 0);
    for (int i = 0; i < C.L; ++i) cnt[R.c[i]]++;
    int64_t nmax = 0;
    for (int k = 0; k < C.q; ++k) if (cnt[k] > nmax) nmax = cnt[k];
    O.n_samples++;
    O.sum_E += R.E;
    unsigned __int128 acc = ((unsigned __int128)(uint64_t)O.sum_E2_hi << 64) | O.sum_E2_lo;
    acc += (unsigned __int128)((__int128)R.E * (__int128)R.E);
    O.sum_E2_lo = (uint64_t)acc;
    O.sum_E2_hi = (int64_t)(uint64_t)(acc >> 64);
    O.sum_Nmax += nmax;
    O.sum_Nmax2 += nmax * nmax;
    // Eq. 11 needs <E^4>: E^4 = (E^2)^2 with E^2 = hi 2^64 + lo, added limb by limb (schoolbook, base 2^64)
    {
        const unsigned __int128 e2 = (unsigned __int128)((__int128)R.E * (__int128)R.E);
        const uint64_t lo = (uint64_t)e2, hi = (uint64_t)(e2 >> 64);
        const unsigned __int128 ll = (unsigned __int128)lo * lo, lh = (unsigned __int128)lo * hi,
                                hh = (unsigned __int128)hi * hi;
        uint64_t add[4] = {(uint64_t)ll, 0, 0, 0};
        unsigned __int128 c = (ll >> 64) + (uint64_t)lh + (uint64_t)lh;     // limb 1: carry of ll + 2 low(lh)
        add[1] = (uint64_t)c;
        c = (c >> 64) + (lh >> 64) + (lh >> 64) + (uint64_t)hh;             // limb 2
        add[2] = (uint64_t)c;
        c = (c >> 64) + (hh >> 64);                                         // limb 3
        add[3] = (uint64_t)c;
        unsigned __int128 carry = 0;
        for (int k = 0; k < 4; ++k) {
            carry += (unsigned __int128)O.sum_E4[k] + add[k];
            O.sum_E4[k] = (uint64_t)carry;
            carry >>= 64;
        }
    }
    // Eq. 12 needs <M^4>, a polynomial in Nmax of degree 4 (Eq. 10)
    O.sum_Nmax3 += nmax * nmax * nmax;
    unsigned __int128 n4 = ((unsigned __int128)(uint64_t)O.sum_Nmax4_hi << 64) | O.sum_Nmax4_lo;
    n4 += (unsigned __int128)((uint64_t)(nmax * nmax)) * (uint64_t)(nmax * nmax);
    O.sum_Nmax4_lo = (uint64_t)n4;
    O.sum_Nmax4_hi = (int64_t)(uint64_t)(n4 >> 64);
}

// Eq. 9 in two stages, even pairs then odd pairs (A11).
void swap_event(Ctx& C, int e) {
    for (int stage = 0; stage < 2; ++stage) {
        for (int t = stage; t + 1 < C.n_rep; t += 2) {
            Replica& Ra = C.rep[(size_t)e * C.n_rep + t];
            Replica& Rb = C.rep[(size_t)e * C.n_rep + t + 1];
            Obs& O = C.obs[(size_t)e * C.n_rep + t];
            const double d = (C.beta[t] - C.beta[t + 1]) * ldexp((double)(Ra.E - Rb.E), -24);
            const uint32_t ctr[4] = {(uint32_t)t, (uint32_t)C.sweep, 0u, ((uint32_t)(C.ens_base + e) << 4) | TAG_SWAP};
            uint32_t w[4];
            philox4x32_10(ctr, C.key, w);
            const double u = uniform53(w[1], w[2]);
            O.swap_attempts++;
            if (d < 0 && fabs(u - exp(d)) < 1e-12) O.near_ties++;
            if (d >= 0 || u < exp(d)) {
                std::swap(Ra.c, Rb.c);      // A12: configurations move between slots
                std::swap(Ra.E, Rb.E);
                std::swap(Ra.h, Rb.h);
                O.swap_accepts++;
            }
        }
    }
}

// Floating-point comparison modes: arith = 1 (fp32) or 2 (fp64).  A context is used in ONE mode from creation (or
// from a point where its running energies are exact: the first call converts E to the floating type).
template <typename T>
int sweeps_float(Ctx& C, int64_t n, int swap_every, int n_threads, bool first) {
    const int R = C.n_ens * C.n_rep;
    std::vector<T> Jf(C.L);
    for (int r = 0; r < C.L; ++r) Jf[r] = (T)ldexp((double)C.Jq[r], -24);
    if (first)
        for (int x = 0; x < R; ++x) C.rep[x].Ef = (double)(T)ldexp((double)C.rep[x].E, -24);
    if (n_threads < 1) n_threads = 1;
    if (n_threads > R) n_threads = R;
    for (int64_t s = 0; s < n; ++s) {
        C.sweep += 1;
        auto work = [&](int tid) {
            for (int x = tid; x < R; x += n_threads) {
                metropolis_cycle_float<T>(C, Jf, x / C.n_rep, x % C.n_rep);
                measure(C, x / C.n_rep, x % C.n_rep);
            }
        };
        if (n_threads == 1) work(0);
        else {
            std::vector<std::thread> th;
            for (int t = 0; t < n_threads; ++t) th.emplace_back(work, t);
            for (auto& t : th) t.join();
        }
        if (swap_every > 0 && C.sweep % swap_every == 0)
            for (int e = 0; e < C.n_ens; ++e) swap_event_float(C, e);
    }
    return 0;
}

}  // namespace

// ---------------------------------------------------------------------------
// C interface (ctypes; oracle/pt_oracle.py).  All pointers are host pointers.
// ---------------------------------------------------------------------------
extern "C" {

// fp64 copy of J*(r), r = 1..L-1 into out[1..L-1]; out[0] = 0.
int orc_jstar(int L, double sigma, double* out) {
    out[0] = 0.0;
    for (int r = 1; r < L; ++r) out[r] = (double)jstar(L, (long double)sigma, r);
    return 0;
}

int orc_couplings(int L, double sigma, int32_t* Jq) {
    std::vector<int32_t> v;
    couplings(L, sigma, v);
    std::memcpy(Jq, v.data(), sizeof(int32_t) * (size_t)L);
    return 0;
}

int orc_philox(const uint32_t* ctr, const uint32_t* key, uint32_t* out) {
    philox4x32_10(ctr, key, out);
    return 0;
}

double orc_uniform53(uint32_t w1, uint32_t w2) { return uniform53(w1, w2); }

// Returns NULL on invalid arguments (same validity rules as include/pt.h).
void* orc_create_ex(int L, int q, double sigma, int n_ens, int n_rep, const double* betas, uint64_t seed,
                    int ens_base) {
    if (ens_base < 0) return nullptr;
    if (L < 2 || (L % 8) != 0 || q < 2 || q > 64 || !(sigma > 0.0) || !std::isfinite(sigma) ||
        n_ens < 1 || n_rep < 1 || !betas)
        return nullptr;
    for (int t = 0; t < n_rep; ++t)
        if (!(betas[t] >= 0.0) || !std::isfinite(betas[t])) return nullptr;
    Ctx* C = new Ctx;
    C->L = L; C->q = q; C->sigma = sigma; C->n_ens = n_ens; C->n_rep = n_rep; C->seed = seed;
    C->ens_base = ens_base;
    C->key[0] = (uint32_t)seed; C->key[1] = (uint32_t)(seed >> 32);
    C->beta.assign(betas, betas + n_rep);
    couplings(L, sigma, C->Jq);
    int64_t rowsum = 0;
    for (int r = 0; r < L; ++r) rowsum += C->Jq[r];
    if (rowsum >= ((int64_t)1 << 31)) { delete C; return nullptr; }
    C->rep.resize((size_t)n_ens * n_rep);
    C->obs.assign((size_t)n_ens * n_rep, Obs{});
    // INIT: hot start, colours uniform in {0..q-1} from Philox (tag INIT, sweep 0)
    for (int e = 0; e < n_ens; ++e)
        for (int t = 0; t < n_rep; ++t) {
            Replica& R = C->rep[(size_t)e * n_rep + t];
            R.c.resize(L);
            for (int i = 0; i < L; ++i) {
                const uint32_t ctr[4] = {(uint32_t)i, 0u, (uint32_t)t, ((uint32_t)(C->ens_base + e) << 4) | TAG_INIT};
                uint32_t w[4];
                philox4x32_10(ctr, C->key, w);
                R.c[i] = (uint8_t)mulhi32(w[0], (uint32_t)q);
            }
            R.E = total_energy(*C, R.c);
        }
    return C;
}

void* orc_create(int L, int q, double sigma, int n_ens, int n_rep, const double* betas, uint64_t seed) {
    return orc_create_ex(L, q, sigma, n_ens, n_rep, betas, seed, 0);
}

void orc_destroy(void* h) { delete (Ctx*)h; }

// n sweeps; swap event when swap_every>0 and sweep % swap_every == 0 (A10).
// field=0: direct O(L) sum per attempt (the paper's way).  field=1: per-colour
// local fields (same integers, checked equal in tests).  n_threads>1: replicas
// of one sweep are distributed over std::threads and joined before the swaps;
// replicas are independent within a sweep, so results are identical.
int orc_sweeps(void* hh, int64_t n, int swap_every, int field, int n_threads) {
    Ctx& C = *(Ctx*)hh;
    if (n < 0 || swap_every < 0) return -1;
    const int R = C.n_ens * C.n_rep;
    if (field)
        for (int x = 0; x < R; ++x) build_fields(C, C.rep[x]);
    if (n_threads < 1) n_threads = 1;
    if (n_threads > R) n_threads = R;
    for (int64_t s = 0; s < n; ++s) {
        C.sweep += 1;
        auto work = [&](int tid) {
            for (int x = tid; x < R; x += n_threads) {
                metropolis_cycle(C, x / C.n_rep, x % C.n_rep, field != 0);
                measure(C, x / C.n_rep, x % C.n_rep);
            }
        };
        if (n_threads == 1) work(0);
        else {
            std::vector<std::thread> th;
            for (int t = 0; t < n_threads; ++t) th.emplace_back(work, t);
            for (auto& t : th) t.join();
        }
        if (swap_every > 0 && C.sweep % swap_every == 0)
            for (int e = 0; e < C.n_ens; ++e) swap_event(C, e);
    }
    if (field)
        for (int x = 0; x < R; ++x) { C.rep[x].h.clear(); C.rep[x].h.shrink_to_fit(); }
    return 0;
}

int orc_sweeps_arith(void* hh, int64_t n, int swap_every, int arith, int n_threads) {
    Ctx& C = *(Ctx*)hh;
    if (n < 0 || swap_every < 0 || (arith != 1 && arith != 2)) return -1;
    const bool first = C.float_mode == 0;
    if (!first && C.float_mode != arith) return -1;
    C.float_mode = arith;
    return arith == 1 ? sweeps_float<float>(C, n, swap_every, n_threads, first)
                      : sweeps_float<double>(C, n, swap_every, n_threads, first);
}

// dE of changing site i of (ens, slot) to colour b_api in the floating-point mode arith (1 fp32, 2 fp64), as a double.
double orc_delta_e_arith(void* hh, int ens, int slot, int i, int b_api, int arith) {
    Ctx& C = *(Ctx*)hh;
    const Replica& R = C.rep[(size_t)ens * C.n_rep + slot];
    if (arith == 1) {
        std::vector<float> Jf(C.L);
        for (int r = 0; r < C.L; ++r) Jf[r] = (float)ldexp((double)C.Jq[r], -24);
        return (double)delta_e_float<float>(C, Jf, R.c, i, R.c[i], b_api - 1);
    }
    std::vector<double> Jf(C.L);
    for (int r = 0; r < C.L; ++r) Jf[r] = ldexp((double)C.Jq[r], -24);
    return delta_e_float<double>(C, Jf, R.c, i, R.c[i], b_api - 1);
}

int orc_energy(void* hh, int64_t* E_out, int recompute) {
    Ctx& C = *(Ctx*)hh;
    for (size_t x = 0; x < C.rep.size(); ++x)
        E_out[x] = recompute ? total_energy(C, C.rep[x].c) : C.rep[x].E;
    return 0;
}

int orc_observables(void* hh, void* out) {
    Ctx& C = *(Ctx*)hh;
    std::memcpy(out, C.obs.data(), sizeof(Obs) * C.obs.size());
    return 0;
}

int orc_get_spins(void* hh, uint8_t* out) {
    Ctx& C = *(Ctx*)hh;
    for (size_t x = 0; x < C.rep.size(); ++x)
        for (int i = 0; i < C.L; ++i) out[x * C.L + i] = (uint8_t)(C.rep[x].c[i] + 1);   // A4: API 1..q
    return 0;
}

int orc_set_spins(void* hh, const uint8_t* in) {
    Ctx& C = *(Ctx*)hh;
    for (size_t x = 0; x < C.rep.size(); ++x)
        for (int i = 0; i < C.L; ++i) {
            const int v = in[x * C.L + i];
            if (v < 1 || v > C.q) return -1;
        }
    for (size_t x = 0; x < C.rep.size(); ++x) {
        for (int i = 0; i < C.L; ++i) C.rep[x].c[i] = (uint8_t)(in[x * C.L + i] - 1);
        C.rep[x].E = total_energy(C, C.rep[x].c);
    }
    return 0;
}

int orc_get_couplings(void* hh, int32_t* Jq) {
    Ctx& C = *(Ctx*)hh;
    std::memcpy(Jq, C.Jq.data(), sizeof(int32_t) * (size_t)C.L);
    return 0;
}

int64_t orc_sweep_counter(void* hh) { return ((Ctx*)hh)->sweep; }

// 0: sequential site order (default), 1: random sites.  The floating-point comparison modes are sequential only.
int orc_set_site_order(void* hh, int order) {
    if (order != 0 && order != 1) return -1;
    ((Ctx*)hh)->site_order = order;
    return 0;
}

// dE of changing site i of (ens, slot) to colour b_api (1..q), by the direct sum.
int64_t orc_delta_e(void* hh, int ens, int slot, int i, int b_api) {
    Ctx& C = *(Ctx*)hh;
    const Replica& R = C.rep[(size_t)ens * C.n_rep + slot];
    return delta_e_direct(C, R.c, i, R.c[i], b_api - 1);
}

int orc_obs_size(void) { return (int)sizeof(Obs); }

}  // extern "C"

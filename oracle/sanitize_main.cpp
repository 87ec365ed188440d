// oracle/sanitize_main.cpp -- TEST INFRASTRUCTURE.  A small driver that exercises every entry point of
// pt_oracle.cpp; tests/test_oracle_sanitize.py links the two with -fsanitize=address,undefined and runs the result
// ("oracle under -fsanitize=address,undefined").  Exit code 0 and an empty sanitizer report
// are the pass criterion; the numbers printed are only there so that nothing is optimised away.
#include <cstdint>
#include <cstdio>
#include <vector>

extern "C" {
int orc_jstar(int L, double sigma, double* out);
int orc_couplings(int L, double sigma, int32_t* Jq);
int orc_philox(const uint32_t* ctr, const uint32_t* key, uint32_t* out);
double orc_uniform53(uint32_t w1, uint32_t w2);
void* orc_create_ex(int L, int q, double sigma, int n_ens, int n_rep, const double* betas, uint64_t seed, int ens_base);
void orc_destroy(void* h);
int orc_sweeps(void* h, int64_t n, int swap_every, int field, int n_threads);
int orc_energy(void* h, int64_t* E_out, int recompute);
int orc_observables(void* h, void* out);
int orc_get_spins(void* h, uint8_t* out);
int orc_set_spins(void* h, const uint8_t* in);
int orc_get_couplings(void* h, int32_t* Jq);
int64_t orc_sweep_counter(void* h);
int64_t orc_delta_e(void* h, int ens, int slot, int i, int b_api);
int orc_obs_size(void);
}

int main() {
    long long check = 0;
    {
        std::vector<double> J(64);
        std::vector<int32_t> Jq(64);
        orc_jstar(64, 0.5, J.data());
        orc_couplings(64, 0.5, Jq.data());
        check += Jq[1] + Jq[32];
        const uint32_t ctr[4] = {1, 2, 3, 4}, key[2] = {5, 6};
        uint32_t w[4];
        orc_philox(ctr, key, w);
        check += (long long)(orc_uniform53(w[1], w[2]) * 1000.0);
    }
    struct Shape { int L, q, n_ens, n_rep; double sigma; };
    const Shape shapes[] = {{8, 2, 1, 1, 0.5}, {64, 3, 2, 5, 0.4}, {40, 16, 1, 3, 0.9}, {128, 8, 1, 4, 0.3}, {48, 37, 1, 2, 0.6}};
    for (const Shape& s : shapes) {
        std::vector<double> betas(s.n_rep);
        for (int t = 0; t < s.n_rep; ++t) betas[t] = 0.3 + 0.4 * t;
        void* h = orc_create_ex(s.L, s.q, s.sigma, s.n_ens, s.n_rep, betas.data(), 0x1308542600000000ull + s.L, 1);
        if (!h) return 2;
        const size_t R = (size_t)s.n_ens * s.n_rep;
        std::vector<int64_t> E(R), E2(R);
        std::vector<uint8_t> spins(R * s.L), obs(R * (size_t)orc_obs_size());
        std::vector<int32_t> Jq(s.L);
        for (int field = 0; field < 2; ++field)
            for (int threads = 1; threads <= 3; threads += 2) {
                if (orc_sweeps(h, 7, 1, field, threads)) return 3;
                if (orc_sweeps(h, 5, 3, field, threads)) return 3;
                if (orc_sweeps(h, 2, 0, field, threads)) return 3;
            }
        orc_energy(h, E.data(), 0);
        orc_energy(h, E2.data(), 1);
        for (size_t x = 0; x < R; ++x) {
            if (E[x] != E2[x]) return 4;   // running energy == O(L^2) recount
            check += E[x];
        }
        orc_observables(h, obs.data());
        orc_get_spins(h, spins.data());
        orc_get_couplings(h, Jq.data());
        check += orc_delta_e(h, 0, 0, s.L - 1, 1 + (spins[s.L - 1] % s.q));
        for (size_t n = 0; n < spins.size(); ++n) spins[n] = (uint8_t)(1 + (n * 7 + 3) % s.q);
        if (orc_set_spins(h, spins.data())) return 5;
        spins[0] = (uint8_t)(s.q + 1);
        if (orc_set_spins(h, spins.data()) == 0) return 6;   // colour out of range must be refused
        if (orc_sweeps(h, -1, 1, 0, 1) == 0) return 7;
        check += orc_sweep_counter(h);
        orc_destroy(h);
    }
    // invalid arguments must be refused, not crash
    const double b1[1] = {1.0};
    if (orc_create_ex(12, 3, 0.5, 1, 1, b1, 1, 0)) return 8;
    if (orc_create_ex(64, 65, 0.5, 1, 1, b1, 1, 0)) return 8;
    if (orc_create_ex(64, 3, 0.5, 1, 1, nullptr, 1, 0)) return 8;
    std::printf("sanitize_main OK %lld\n", check);
    return 0;
}

// pt_lib.cu -- host side of libpt (C ABI in include/pt.h) for sm_100a.
// Validates arguments, owns the device state of a context and enqueues the
// kernels of pt_kernels.cuh / pt_sweep_*.cuh.  There is no CPU fallback: every
// step of the path (J* table, hot start, energies, sweeps, swaps, observables)
// runs in the kernels; without a CUDA device every call fails with PT_ECUDA.
#include <cuda_runtime.h>

#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <string>
#include <vector>
#include <algorithm>

#include "pt.h"
#include "pt_kernels.cuh"
#include "pt_sweep_direct.cuh"
#include "pt_sweep_field.cuh"
#include "pt_peaks.cuh"
#include "pt_sweep_float.cuh"

namespace {

thread_local std::string g_err;

int fail(int code, const std::string& msg) {
    g_err = msg;
    return code;
}

#define PT_CUDA(call)                                                                      \
    do {                                                                                   \
        cudaError_t err__ = (call);                                                        \
        if (err__ != cudaSuccess)                                                          \
            return fail(err__ == cudaErrorMemoryAllocation ? PT_ENOMEM : PT_ECUDA,         \
                        std::string(#call) + ": " + cudaGetErrorString(err__));            \
    } while (0)

constexpr size_t kSmemLimit = 227 * 1024;  // per CTA on sm_100

// Every entry point runs on the context's device, whatever the caller's current device is, and restores it.
struct DeviceGuard {
    int prev = -1, want = -1;
    explicit DeviceGuard(int dev) : want(dev) {
        if (cudaGetDevice(&prev) != cudaSuccess) prev = -1;
        if (prev != want) cudaSetDevice(want);
    }
    ~DeviceGuard() {
        if (prev >= 0 && prev != want) cudaSetDevice(prev);
    }
    DeviceGuard(const DeviceGuard&) = delete;
    DeviceGuard& operator=(const DeviceGuard&) = delete;
};

}  // namespace

struct pt_ctx {
    int L = 0, q = 0, n_ens = 0, n_rep = 0, ens_base = 0;
    double sigma = 0;
    uint64_t seed = 0;
    int device = 0;
    cudaStream_t stream = nullptr;
    int variant = PT_VARIANT_FIELD;
    bool fields_valid = false;
    int64_t sweep = 0;
    long long rowsum = 0;  // sum_r Jq[r]
    int rep_base = 0, n_local = 0;   // slot-sharded context: local storage indices (n_local = 0: not sharded)
    int r_hi = 0;  // largest r <= L/2 with Jq[r] >= 2^16 (direct variant: reach of the high halves)
    int far_ok = 0;  // L = 4096: every far j-range of the direct kernel fits 8-bit residuals (pt_sweep_direct.cuh, FAR)
    int32_t* d_Jq = nullptr;
    uint32_t* d_Jpair = nullptr;
    double* d_beta = nullptr;
    double* d_scale = nullptr;
    uint32_t* d_spins = nullptr;
    long long* d_E = nullptr;
    long long* d_Etmp = nullptr;
    long long* d_Eout = nullptr;
    int* d_perm = nullptr;
    pt_obs* d_obs = nullptr;
    int32_t* d_h = nullptr;
    unsigned* d_done = nullptr;
    int* d_flag = nullptr;
    long long* d_dbg = nullptr;
    unsigned* d_gen = nullptr;
    long long* d_Epub = nullptr;
    uint8_t* d_stage = nullptr;   // [R*L] one byte per spin: staging for pt_get_spins / pt_set_spins / pt_set_state
    uint8_t* h_stage = nullptr;   // pinned host bounce buffer of the same size
    int site_order = 0;      // PT_ORDER_SEQUENTIAL | PT_ORDER_RANDOM (field variant only)
    double* d_Ef = nullptr;  // floating-point comparison variants: running energies in units of 1, storage order
    bool ef_valid = false;   // d_Ef continues the running energies (else it is set from d_E at the next float launch)
    int* h_err = nullptr;    // pinned, device-mapped flag: an in-kernel barrier timed out
    int* d_err = nullptr;    // its device address
    int coresident = -1;   // direct variant: CTAs that fit on the device at once (-1: not asked yet)
    ptk::direct_kernel_t direct_kern = nullptr;   // the sweep kernel instantiation this context uses
    int persistent_policy = 1;   // 0 never, 1 when the context fills the device and the call is long enough, 2 whenever possible

    int R() const { return n_ens * n_rep; }
    int bits() const { return q <= 16 ? 4 : 8; }     // bits per spin in d_spins
    int words() const { return L * bits() / 32; }    // 32-bit words per configuration
    ptk::Dev dev() const {
        ptk::Dev d;
        d.bits = bits(); d.L = L; d.W = words(); d.q = q; d.n_ens = n_ens; d.n_rep = n_rep; d.ens_base = ens_base;
        d.key0 = (uint32_t)seed; d.key1 = (uint32_t)(seed >> 32); d.rowsum = (uint32_t)rowsum;
        d.Jq = d_Jq; d.Jpair = d_Jpair; d.beta = d_beta; d.thr_scale = d_scale;
        d.spins = d_spins; d.E = d_E; d.perm = d_perm; d.obs = d_obs; d.h = d_h; d.done = d_done; d.dbg = d_dbg; d.gen = d_gen; d.Epub = d_Epub; d.err = d_err;
        d.rep_base = rep_base; d.n_local = n_local ? n_local : n_rep; d.count_swaps = rep_base == 0 ? 1 : 0;
        d.far = far_ok;
        return d;
    }
};

namespace {

bool field_fits(int L, int q) { return ptk::field_smem_bytes(L, q) + 512 <= kSmemLimit; }
// Local-field variant over a thread-block cluster (sweep_field_cluster_kernel): can C CTAs hold the replica?
bool field_cluster_fits(int L, int q, int C) {
    return ptk::field_cluster_divides(L, C) && ptk::field_cluster_smem_bytes(L, q, C) + 4096 <= kSmemLimit;
}
// Smallest portable cluster size (2, 4, 8) whose CTAs hold the local fields of one replica; 0 if none does.
int field_cluster_size(int L, int q) {
    for (int C = 2; C <= ptk::FIELD_CLUSTER_MAX; C *= 2)
        if (field_cluster_fits(L, q, C)) return C;
    return 0;
}
bool direct_applies(int L, int q) { return ptk::direct_applies(L, q); }

void free_ctx(pt_ctx* c) {
    if (!c) return;
    cudaFree(c->d_Jq); cudaFree(c->d_Jpair); cudaFree(c->d_beta); cudaFree(c->d_scale);
    cudaFree(c->d_spins); cudaFree(c->d_E); cudaFree(c->d_Etmp); cudaFree(c->d_Eout);
    cudaFree(c->d_perm); cudaFree(c->d_obs); cudaFree(c->d_h); cudaFree(c->d_done); cudaFree(c->d_flag); cudaFree(c->d_dbg); cudaFree(c->d_gen); cudaFree(c->d_Epub);
    if (c->h_err) cudaFreeHost(c->h_err);
    cudaFree(c->d_stage);
    cudaFree(c->d_Ef);
    if (c->h_stage) cudaFreeHost(c->h_stage);
    delete c;
}

int recompute_energy(pt_ctx* c, long long* d_out) {
    if (ptk::energy_direct_applies(c->L, c->q)) {   // IDP.2A version (pt_sweep_direct.cuh), ~10x faster at L = 4096
        int rc = ptk::launch_energy_direct(c->dev(), d_out, c->stream);
        if (rc) return fail(PT_ECUDA, std::string("energy_direct launch: ") + cudaGetErrorString((cudaError_t)rc));
        return PT_OK;
    }
    const size_t smem = (size_t)(c->L + c->words()) * 4;
    if (smem > 48 * 1024) PT_CUDA((cudaError_t)ptk::allow_max_dynamic_smem((const void*)ptk::energy_kernel, 1024));
    ptk::energy_kernel<<<c->R(), 256, smem, c->stream>>>(c->dev(), d_out);
    PT_CUDA(cudaGetLastError());
    return PT_OK;
}

int ensure_fields(pt_ctx* c) {
    if (c->fields_valid) return PT_OK;
    if (!c->d_h) PT_CUDA(cudaMalloc(&c->d_h, (size_t)c->R() * c->q * c->L * sizeof(int32_t)));
    const size_t smem = (size_t)(c->L + c->words()) * 4;
    if (smem > 48 * 1024) PT_CUDA((cudaError_t)ptk::allow_max_dynamic_smem((const void*)ptk::build_fields_kernel, 1024));
    ptk::build_fields_kernel<<<c->R(), 256, smem, c->stream>>>(c->dev());
    PT_CUDA(cudaGetLastError());
    c->fields_valid = true;
    return PT_OK;
}

// Cluster size the local-field sweep of this context runs with (0: one CTA per replica).  A replica whose fields do
// not fit in one SM takes the smallest cluster that holds them; PT_FIELD_CLUSTER=2|4|8 (tests, measurements) asks
// for a cluster also where one CTA would do.  Sequential site order only.
int field_cluster_of(const pt_ctx* c) {
    if (c->site_order == PT_ORDER_RANDOM) return 0;
    const char* env = getenv("PT_FIELD_CLUSTER");
    if (env && env[0] >= '2' && env[0] <= '8' && env[1] == 0) {
        const int C = env[0] - '0';
        if ((C == 2 || C == 4 || C == 8) && field_cluster_fits(c->L, c->q, C)) return C;
    }
    return field_fits(c->L, c->q) ? 0 : field_cluster_size(c->L, c->q);
}

// rowsum = sum_r Jq[r]: the direct variant keeps theta - dE in int32 and needs |dE| <= rowsum < 2^30 - 1.
int resolve_variant(int L, int q, long long rowsum, int variant, int* out) {
    const bool direct_ok = direct_applies(L, q) && rowsum < (1ll << 30) - 1;
    if (variant == PT_VARIANT_AUTO) variant = direct_ok ? PT_VARIANT_DIRECT : PT_VARIANT_FIELD;
    if (variant == PT_VARIANT_DIRECT) {
        if (!direct_ok)
            return fail(PT_EINVAL, "direct variant needs L % 64 == 0, 64 <= L <= 10240 (L <= 9664 for q > 8: shared memory) "
                                   "and sum_r Jq[r] < 2^30 - 1");
    } else if (variant == PT_VARIANT_FIELD) {
        if (!field_fits(L, q) && !field_cluster_size(L, q))
            return fail(PT_ECAPACITY, "local-field table (L*q*4 bytes) does not fit in the shared memory of a cluster of 8 SMs");
    } else if (variant == PT_VARIANT_FP32 || variant == PT_VARIANT_FP64) {
        const size_t smem = variant == PT_VARIANT_FP32 ? ptk::float_smem_bytes<float>(L) : ptk::float_smem_bytes<double>(L);
        if (smem + 2048 > kSmemLimit) return fail(PT_ECAPACITY, "couplings and uniforms (L*14 or L*18 bytes) do not fit in shared memory");
    } else {
        return fail(PT_EINVAL, "unknown variant");
    }
    *out = variant;
    return PT_OK;
}

// Enqueue one launch covering n_sweeps sweeps.  swap_mode 0: no swap event, 1: one at the end of the launch,
// 2 (direct variant only): persistent launch with an event after every sweep whose index divides by swap_every.
int launch_sweeps(pt_ctx* c, int n_sweeps, int swap_mode, int swap_every) {
    if (c->variant == PT_VARIANT_FIELD) {
        int rc = ensure_fields(c);
        if (rc) return rc;
    }
    const ptk::Dev d = c->dev();  // after ensure_fields: it may allocate d_h
    if (c->variant == PT_VARIANT_FP32 || c->variant == PT_VARIANT_FP64) {
        const bool f32 = c->variant == PT_VARIANT_FP32;
        if (!c->d_Ef) PT_CUDA(cudaMalloc(&c->d_Ef, (size_t)c->R() * sizeof(double)));
        if (!c->ef_valid) {   // entering the variant: the running energies are exact integers
            if (f32) ptk::energy_to_float_kernel<float><<<(c->R() + 255) / 256, 256, 0, c->stream>>>(d, c->d_Ef);
            else ptk::energy_to_float_kernel<double><<<(c->R() + 255) / 256, 256, 0, c->stream>>>(d, c->d_Ef);
            PT_CUDA(cudaGetLastError());
            c->ef_valid = true;
        }
        c->fields_valid = false;
        if (f32) {
            PT_CUDA((cudaError_t)ptk::allow_max_dynamic_smem((const void*)ptk::sweep_float_kernel<float>, 2048));
            ptk::sweep_float_kernel<float><<<c->R(), ptk::FLOAT_THREADS, ptk::float_smem_bytes<float>(c->L), c->stream>>>(
                d, c->d_Ef, (long long)c->sweep, n_sweeps, swap_mode == 1 ? 1 : 0);
        } else {
            PT_CUDA((cudaError_t)ptk::allow_max_dynamic_smem((const void*)ptk::sweep_float_kernel<double>, 2048));
            ptk::sweep_float_kernel<double><<<c->R(), ptk::FLOAT_THREADS, ptk::float_smem_bytes<double>(c->L), c->stream>>>(
                d, c->d_Ef, (long long)c->sweep, n_sweeps, swap_mode == 1 ? 1 : 0);
        }
    } else if (c->variant == PT_VARIANT_FIELD && field_cluster_of(c) > 0) {
        // one thread-block cluster per replica: the local fields are spread over the shared memory of C SMs
        const int C = field_cluster_of(c);
        typedef void (*field_kernel_t)(ptk::Dev, long long, int, int);
        const field_kernel_t kern = c->bits() == 8 ? ptk::sweep_field_cluster_kernel<8> : ptk::sweep_field_cluster_kernel<4>;
        PT_CUDA((cudaError_t)ptk::allow_max_dynamic_smem((const void*)kern, 4096));
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3((unsigned)(c->R() * C));
        cfg.blockDim = dim3((unsigned)ptk::FIELD_THREADS);
        cfg.dynamicSmemBytes = ptk::field_cluster_smem_bytes(c->L, c->q, C);
        cfg.stream = c->stream;
        cudaLaunchAttribute attr[1];
        attr[0].id = cudaLaunchAttributeClusterDimension;
        attr[0].val.clusterDim.x = (unsigned)C;
        attr[0].val.clusterDim.y = 1;
        attr[0].val.clusterDim.z = 1;
        cfg.attrs = attr;
        cfg.numAttrs = 1;
        PT_CUDA(cudaLaunchKernelEx(&cfg, kern, d, (long long)c->sweep, n_sweeps, swap_mode == 1 ? 1 : 0));
    } else if (c->variant == PT_VARIANT_FIELD) {
        const size_t smem = ptk::field_smem_bytes(c->L, c->q, c->site_order == PT_ORDER_RANDOM);
        typedef void (*field_kernel_t)(ptk::Dev, long long, int, int);
        const bool rnd = c->site_order == PT_ORDER_RANDOM, wide = c->bits() == 8;
        const field_kernel_t kern = rnd ? (wide ? ptk::sweep_field_kernel<true, 8> : ptk::sweep_field_kernel<true, 4>)
                                        : (wide ? ptk::sweep_field_kernel<false, 8> : ptk::sweep_field_kernel<false, 4>);
        PT_CUDA((cudaError_t)ptk::allow_max_dynamic_smem((const void*)kern, 1024));
        kern<<<c->R(), ptk::FIELD_THREADS, smem, c->stream>>>(d, (long long)c->sweep, n_sweeps, swap_mode == 1 ? 1 : 0);
    } else {
        c->fields_valid = false;
        if (!c->direct_kern) c->direct_kern = ptk::select_direct_kernel(d, c->r_hi, c->device, &c->coresident);
        int rc = ptk::launch_sweep_direct(c->direct_kern, d, (long long)c->sweep, n_sweeps, swap_mode, swap_every,
                                          c->r_hi, c->stream);
        if (rc) return fail(PT_ECUDA, std::string("sweep_direct launch: ") + cudaGetErrorString((cudaError_t)rc));
    }
    PT_CUDA(cudaGetLastError());
    c->sweep += n_sweeps;
    return PT_OK;
}

// Direct variant: can all replicas be resident at once (persistent launches with in-kernel swap events)?
bool persistent_ok(pt_ctx* c) {
    if (c->variant != PT_VARIANT_DIRECT || c->persistent_policy == 0 || c->n_local) return false;
    if (!c->direct_kern) c->direct_kern = ptk::select_direct_kernel(c->dev(), c->r_hi, c->device, &c->coresident);
    // A small context (e.g. one of the 40 handles of configs[4]) shares the GPU with others: launches per swap
    // interval interleave their CTAs better than resident kernels that wait at their own barriers (measured:
    // 4.2e9 against 3.6e9 attempts/s on configs[4]).  Persistent launches are for contexts that take at least a
    // third of the SMs (configs[2] alone: 32 us per sweep persistent, 39 us with ordinary launches).
    int n_sm = 0;
    if (cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, c->device) != cudaSuccess) return false;
    return c->R() <= c->coresident && (3 * c->R() >= n_sm || c->persistent_policy == 2) &&
           c->n_rep <= ptk::DIRECT_MAX_PERSIST_REP;
}

}  // namespace

extern "C" {

const char* pt_last_error(void) { return g_err.c_str(); }

int pt_create_ex(pt_ctx** out, int L, int q, double sigma, int n_ens, int n_rep, const double* betas,
                 uint64_t seed, int ens_base) {
    if (!out) return fail(PT_EINVAL, "out is NULL");
    *out = nullptr;
    if (L < 8 || (L % 8) != 0) return fail(PT_EINVAL, "L must be >= 8 and a multiple of 8");
    if (L > (1 << 20)) return fail(PT_EINVAL, "L too large");
    if (q < 2 || q > ptk::PT_QMAX) return fail(PT_EINVAL, "q must be in 2..64");
    if (!(sigma > 0.0) || !std::isfinite(sigma)) return fail(PT_EINVAL, "sigma must be finite and > 0");
    if (n_ens < 1 || n_rep < 1) return fail(PT_EINVAL, "n_ens and n_rep must be >= 1");
    if ((long long)n_ens * n_rep > (1 << 24)) return fail(PT_EINVAL, "too many replicas");
    if (ens_base < 0 || (long long)ens_base + n_ens > (1ll << 28)) return fail(PT_EINVAL, "ens_base out of range");
    if (!betas) return fail(PT_EINVAL, "betas is NULL");
    for (int t = 0; t < n_rep; ++t)
        if (!(betas[t] >= 0.0) || !std::isfinite(betas[t])) return fail(PT_EINVAL, "betas must be finite and >= 0");

    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
        cudaGetLastError();
        return fail(PT_ECUDA, "no CUDA device: libpt has no CPU path");
    }
    int dev = 0;
    PT_CUDA(cudaGetDevice(&dev));
    cudaDeviceProp prop;
    PT_CUDA(cudaGetDeviceProperties(&prop, dev));
    if (prop.major != 10) return fail(PT_ECUDA, "libpt is built for sm_100a (B200) only");

    int variant = 0;
    {
        int rc = resolve_variant(L, q, 0, PT_VARIANT_AUTO, &variant);
        if (rc) return rc;
    }

    pt_ctx* c = new (std::nothrow) pt_ctx;
    if (!c) return fail(PT_ENOMEM, "host allocation failed");
    c->L = L; c->q = q; c->sigma = sigma; c->n_ens = n_ens; c->n_rep = n_rep; c->seed = seed;
    c->ens_base = ens_base; c->device = dev; c->variant = variant;
    const int R = c->R();
    const int W = q <= 16 ? L / 8 : L / 4;

#define PT_CUDA_C(call)                                                                                   \
    do {                                                                                                  \
        cudaError_t err__ = (call);                                                                       \
        if (err__ != cudaSuccess) {                                                                       \
            free_ctx(c);                                                                                  \
            return fail(err__ == cudaErrorMemoryAllocation ? PT_ENOMEM : PT_ECUDA,                        \
                        std::string(#call) + ": " + cudaGetErrorString(err__));                           \
        }                                                                                                 \
    } while (0)

    PT_CUDA_C(cudaMalloc(&c->d_Jq, (size_t)L * sizeof(int32_t)));
    PT_CUDA_C(cudaMalloc(&c->d_Jpair, (size_t)2 * L * sizeof(uint32_t)));
    PT_CUDA_C(cudaMalloc(&c->d_beta, (size_t)n_rep * sizeof(double)));
    PT_CUDA_C(cudaMalloc(&c->d_scale, (size_t)n_rep * sizeof(double)));
    PT_CUDA_C(cudaMalloc(&c->d_spins, (size_t)R * W * sizeof(uint32_t)));
    PT_CUDA_C(cudaMalloc(&c->d_E, (size_t)R * sizeof(long long)));
    PT_CUDA_C(cudaMalloc(&c->d_Etmp, (size_t)R * sizeof(long long)));
    PT_CUDA_C(cudaMalloc(&c->d_Eout, (size_t)R * sizeof(long long)));
    PT_CUDA_C(cudaMalloc(&c->d_perm, (size_t)R * sizeof(int)));
    PT_CUDA_C(cudaMalloc(&c->d_obs, (size_t)R * sizeof(pt_obs)));
    PT_CUDA_C(cudaMalloc(&c->d_done, (size_t)n_ens * sizeof(unsigned)));
    PT_CUDA_C(cudaMalloc(&c->d_flag, sizeof(int)));
    PT_CUDA_C(cudaMemset(c->d_obs, 0, (size_t)R * sizeof(pt_obs)));
    PT_CUDA_C(cudaMemset(c->d_done, 0, (size_t)n_ens * sizeof(unsigned)));
    PT_CUDA_C(cudaMalloc(&c->d_gen, (size_t)n_ens * sizeof(unsigned)));
    PT_CUDA_C(cudaMemset(c->d_gen, 0, (size_t)n_ens * sizeof(unsigned)));
    PT_CUDA_C(cudaMalloc(&c->d_Epub, (size_t)2 * R * sizeof(long long)));
    PT_CUDA_C(cudaMalloc(&c->d_stage, (size_t)R * L));
    PT_CUDA_C(cudaHostAlloc(&c->h_stage, (size_t)R * L, cudaHostAllocDefault));
    PT_CUDA_C(cudaHostAlloc(&c->h_err, sizeof(int), cudaHostAllocMapped));
    *c->h_err = 0;
    PT_CUDA_C(cudaHostGetDevicePointer(&c->d_err, c->h_err, 0));
    {
        // PT_PERSISTENT=0: one launch per swap interval; =2: persistent launches whenever all replicas can be
        // co-resident (tests); default: only for contexts that fill the device (see persistent_ok)
        const char* env = getenv("PT_PERSISTENT");
        c->persistent_policy = (env && env[0] == '0') ? 0 : (env && env[0] == '2') ? 2 : 1;
    }
#ifdef PT_TIMING
    PT_CUDA_C(cudaMalloc(&c->d_dbg, (size_t)R * 32 * 8 * sizeof(long long)));
    PT_CUDA_C(cudaMemset(c->d_dbg, 0, (size_t)R * 32 * 8 * sizeof(long long)));
#endif

    std::vector<double> scale(n_rep);
    for (int t = 0; t < n_rep; ++t) scale[t] = betas[t] > 0.0 ? 16777216.0 / betas[t] : INFINITY;
    PT_CUDA_C(cudaMemcpy(c->d_beta, betas, (size_t)n_rep * sizeof(double), cudaMemcpyHostToDevice));
    PT_CUDA_C(cudaMemcpy(c->d_scale, scale.data(), (size_t)n_rep * sizeof(double), cudaMemcpyHostToDevice));

    // a1: couplings
    ptk::jstar_kernel<<<(L / 2 + 128) / 128, 128>>>(L, sigma, c->d_Jq, nullptr);
    PT_CUDA_C(cudaGetLastError());
    std::vector<int32_t> Jq(L);
    PT_CUDA_C(cudaMemcpy(Jq.data(), c->d_Jq, (size_t)L * sizeof(int32_t), cudaMemcpyDeviceToHost));
    long long rowsum = 0;
    bool bad = false;
    for (int r = 0; r < L; ++r) { rowsum += Jq[r]; bad |= Jq[r] < 0; }
    for (int r = 1; r <= L / 2; ++r)
        if (Jq[r] >= 65536) c->r_hi = r;
    c->rowsum = rowsum;
    if (L == 4096 && getenv("PT_FAR") && getenv("PT_FAR")[0] == '1') {   // opt-in: measured slower than the plain form
        // FAR: the far half of bulk thread (g, jr) holds Jq[r], r = R0 - 45 .. R0 (mod L), R0 = gbase + 14 - (1024 + 32 jr):
        // it needs max - min <= 255 and 0 < min < 2^15 for every thread
        bool ok = true;
        for (int jr = 0; jr < 64 && ok; ++jr)
            for (int g = 0; g < 4 && ok; ++g) {
                const int gbase = 16 * (g >> 1) + (g & 1);
                const int R0 = ((gbase + 14 - (1024 + 32 * jr)) % L + L) % L;
                int lo = INT32_MAX, hi = 0;
                for (int n = 0; n < 46; ++n) {
                    const int v = Jq[((R0 - n) % L + L) % L];
                    lo = std::min(lo, v); hi = std::max(hi, v);
                }
                ok = hi - lo <= 255 && lo < 32768 && lo > 0;
            }
        c->far_ok = ok ? 1 : 0;
    }
    {
        // PT_VARIANT=direct|field|auto overrides the default choice (an impossible request is an error)
        int want = PT_VARIANT_AUTO;
        const char* env = getenv("PT_VARIANT");
        if (env && !strcmp(env, "direct")) want = PT_VARIANT_DIRECT;
        else if (env && !strcmp(env, "field")) want = PT_VARIANT_FIELD;
        int rc = resolve_variant(L, q, rowsum, want, &c->variant);
        if (rc) { free_ctx(c); return rc; }
    }
    if (bad || rowsum >= (1ll << 31)) {
        free_ctx(c);
        return fail(PT_EOVERFLOW, "sum_r Jq[r] >= 2^31: sigma too small for int32 energy differences");
    }
    ptk::pack_pairs_kernel<<<(L / 2 + 127) / 128, 128>>>(L, c->d_Jq, c->d_Jpair);
    PT_CUDA_C(cudaGetLastError());

    // a2: hot start, permutation, energies
    const ptk::Dev d = c->dev();
    const long long nwords = (long long)R * W;
    ptk::init_spins_kernel<<<(unsigned)((nwords + 255) / 256), 256>>>(d);
    PT_CUDA_C(cudaGetLastError());
    ptk::init_perm_kernel<<<(R + 255) / 256, 256>>>(d);
    PT_CUDA_C(cudaGetLastError());
    {
        int rc = recompute_energy(c, c->d_E);
        if (rc) { free_ctx(c); return rc; }
    }
    PT_CUDA_C(cudaDeviceSynchronize());
#undef PT_CUDA_C
    *out = c;
    return PT_OK;
}

int pt_create(pt_ctx** out, int L, int q, double sigma, int n_ens, int n_rep, const double* betas,
              uint64_t seed) {
    return pt_create_ex(out, L, q, sigma, n_ens, n_rep, betas, seed, 0);
}

void pt_destroy(pt_ctx* ctx) {
    if (!ctx) return;
    DeviceGuard guard(ctx->device);
    cudaStreamSynchronize(ctx->stream);
    free_ctx(ctx);
}

int pt_sweeps_async(pt_ctx* c, int64_t n, int swap_every, int64_t* n_launches) {
    if (!c) return fail(PT_EINVAL, "ctx is NULL");
    DeviceGuard guard(c->device);
    if (n < 0 || swap_every < 0) return fail(PT_EINVAL, "n and swap_every must be >= 0");
    if (c->n_local && swap_every != 0)
        return fail(PT_EINVAL, "slot-sharded context: call pt_sweeps with swap_every = 0 and pt_swap_external");
    // the sweep index is one 32-bit word of the Philox counter (site, sweep, slot, ensemble|tag): beyond 2^32 - 1 sweeps
    // the random streams would repeat
    if (c->sweep + n > 0xffffffffll) return fail(PT_EOVERFLOW, "sweep counter would exceed 2^32 - 1");
    int64_t launches = 0;
    constexpr int64_t kMaxChunk = 1 << 16;  // sweeps per launch
    // a persistent launch pays a counter reset and a cooperative launch: taken for every call of two or more sweeps
    // (single-sweep calls are what interleaved multi-handle drivers issue; they stay ordinary launches)
    const bool persistent = swap_every > 0 && (n >= 2 || c->persistent_policy == 2) && persistent_ok(c);
    while (n > 0) {
        int64_t chunk = n < kMaxChunk ? n : kMaxChunk;
        int swap_mode = c->n_local ? 3 : 0;
        if (persistent) {
            swap_mode = 2;
        } else if (swap_every > 0) {
            const int64_t to_event = swap_every - (c->sweep % swap_every);
            if (to_event <= chunk) { chunk = to_event; swap_mode = 1; }
        }
        if (swap_mode == 2) PT_CUDA(cudaMemsetAsync(c->d_gen, 0, (size_t)c->n_ens * sizeof(unsigned), c->stream));
        int rc = launch_sweeps(c, (int)chunk, swap_mode, swap_every);
        if (rc) return rc;
        launches += 1;
        n -= chunk;
    }
    if (n_launches) *n_launches = launches;
    return PT_OK;
}

int pt_sync(pt_ctx* c) {
    if (!c) return fail(PT_EINVAL, "ctx is NULL");
    DeviceGuard guard(c->device);
    PT_CUDA(cudaStreamSynchronize(c->stream));
    PT_CUDA(cudaGetLastError());
    if (c->h_err && *(volatile int*)c->h_err == 2)
        return fail(PT_ECUDA, "PT_PARANOID: the accept mask of a block differs from its site-by-site forward substitution");
    if (c->h_err && *(volatile int*)c->h_err)
        return fail(PT_ECUDA, "an in-kernel swap barrier timed out (a CTA of the ensemble did not arrive within 30 s): "
                              "the state of this context is lost");
    return PT_OK;
}

int pt_sweeps(pt_ctx* c, int64_t n, int swap_every) {
    int rc = pt_sweeps_async(c, n, swap_every, nullptr);
    if (rc) return rc;
    return pt_sync(c);
}

int pt_energy_dev(pt_ctx* c, int64_t* E_out_dev, int recompute) {
    if (!c || !E_out_dev) return fail(PT_EINVAL, "NULL argument");
    DeviceGuard guard(c->device);
    const long long* src = c->d_E;
    if (recompute) {
        int rc = recompute_energy(c, c->d_Etmp);
        if (rc) return rc;
        src = c->d_Etmp;
    }
    ptk::gather_slots_kernel<<<(c->R() + 255) / 256, 256, 0, c->stream>>>(c->dev(), src, (long long*)E_out_dev);
    PT_CUDA(cudaGetLastError());
    return pt_sync(c);
}

int pt_energy(pt_ctx* c, int64_t* E_out, int recompute) {
    if (!c || !E_out) return fail(PT_EINVAL, "NULL argument");
    DeviceGuard guard(c->device);
    int rc = pt_energy_dev(c, (int64_t*)c->d_Eout, recompute);
    if (rc) return rc;
    PT_CUDA(cudaMemcpy(E_out, c->d_Eout, (size_t)c->R() * sizeof(int64_t), cudaMemcpyDeviceToHost));
    return PT_OK;
}

int pt_observables(pt_ctx* c, pt_obs* out) {
    if (!c || !out) return fail(PT_EINVAL, "NULL argument");
    DeviceGuard guard(c->device);
    int rc = pt_sync(c);
    if (rc) return rc;
    PT_CUDA(cudaMemcpy(out, c->d_obs, (size_t)c->R() * sizeof(pt_obs), cudaMemcpyDeviceToHost));
    for (int x = 0; x < c->R(); ++x) out[x].near_ties = -1;
    return PT_OK;
}

int pt_get_spins_dev(pt_ctx* c, uint8_t* out_dev) {
    if (!c || !out_dev) return fail(PT_EINVAL, "NULL argument");
    DeviceGuard guard(c->device);
    const long long nwords = (long long)c->R() * c->words();
    ptk::unpack_spins_kernel<<<(unsigned)((nwords + 255) / 256), 256, 0, c->stream>>>(c->dev(), out_dev);
    PT_CUDA(cudaGetLastError());
    return pt_sync(c);
}

int pt_get_spins(pt_ctx* c, uint8_t* out) {
    if (!c || !out) return fail(PT_EINVAL, "NULL argument");
    DeviceGuard guard(c->device);
    const size_t n = (size_t)c->R() * c->L;
    int rc = pt_get_spins_dev(c, c->d_stage);
    if (rc) return rc;
    PT_CUDA(cudaMemcpyAsync(c->h_stage, c->d_stage, n, cudaMemcpyDeviceToHost, c->stream));   // pinned: one DMA
    PT_CUDA(cudaStreamSynchronize(c->stream));
    memcpy(out, c->h_stage, n);
    return PT_OK;
}

namespace {
// Uploads n_ens*n_rep*L colours 1..q (host, slot order), checks them and packs them into the spin words.  The state is
// unchanged if a colour is out of range.  Leaves the stream busy (no synchronisation after the pack kernel).
int upload_spins(pt_ctx* c, const uint8_t* in) {
    const size_t n = (size_t)c->R() * c->L;
    memcpy(c->h_stage, in, n);
    PT_CUDA(cudaMemcpyAsync(c->d_stage, c->h_stage, n, cudaMemcpyHostToDevice, c->stream));
    PT_CUDA(cudaMemsetAsync(c->d_flag, 0, sizeof(int), c->stream));
    ptk::check_spins_kernel<<<(unsigned)((n + 255) / 256), 256, 0, c->stream>>>(c->dev(), c->d_stage, c->d_flag);
    PT_CUDA(cudaGetLastError());
    int flag = 0;
    PT_CUDA(cudaMemcpyAsync(&flag, c->d_flag, sizeof(int), cudaMemcpyDeviceToHost, c->stream));
    PT_CUDA(cudaStreamSynchronize(c->stream));
    if (flag) return fail(PT_EINVAL, "colour outside 1..q");
    const long long nwords = (long long)c->R() * c->words();
    ptk::pack_spins_kernel<<<(unsigned)((nwords + 255) / 256), 256, 0, c->stream>>>(c->dev(), c->d_stage);
    PT_CUDA(cudaGetLastError());
    c->fields_valid = false;
    c->ef_valid = false;
    return PT_OK;
}
}  // namespace

int pt_set_spins(pt_ctx* c, const uint8_t* in) {
    if (!c || !in) return fail(PT_EINVAL, "NULL argument");
    DeviceGuard guard(c->device);
    int rc = upload_spins(c, in);
    if (rc) return rc;
    rc = recompute_energy(c, c->d_E);
    if (rc) return rc;
    return pt_sync(c);
}

int pt_get_state(pt_ctx* c, uint8_t* spins, int64_t* E, pt_obs* obs, int64_t* sweep) {
    if (!c || !spins || !E || !obs || !sweep) return fail(PT_EINVAL, "NULL argument");
    if (c->n_local) return fail(PT_EINVAL, "pt_get_state is not available for slot-sharded contexts");
    int rc = pt_get_spins(c, spins);
    if (rc == PT_OK) rc = pt_energy(c, E, 0);
    if (rc == PT_OK) rc = pt_observables(c, obs);
    if (rc == PT_OK) *sweep = c->sweep;
    return rc;
}

int pt_set_state(pt_ctx* c, const uint8_t* spins, const int64_t* E, const pt_obs* obs, int64_t sweep) {
    if (!c || !spins) return fail(PT_EINVAL, "NULL argument");
    if (c->n_local) return fail(PT_EINVAL, "pt_set_state is not available for slot-sharded contexts");
    if (sweep < 0 || sweep > 0xffffffffll) return fail(PT_EINVAL, "sweep counter must be in 0 .. 2^32 - 1");
    DeviceGuard guard(c->device);
    int rc = upload_spins(c, spins);
    if (rc) return rc;
    if (E) {   // the caller's running energies (slot order) -> storage order, no O(L^2) recount
        PT_CUDA(cudaMemcpyAsync(c->d_Eout, E, (size_t)c->R() * sizeof(int64_t), cudaMemcpyHostToDevice, c->stream));
        ptk::scatter_slots_kernel<<<(c->R() + 255) / 256, 256, 0, c->stream>>>(c->dev(), c->d_Eout, c->d_E);
        PT_CUDA(cudaGetLastError());
    } else {
        rc = recompute_energy(c, c->d_E);
        if (rc) return rc;
    }
    if (obs) {
        std::vector<pt_obs> tmp(obs, obs + c->R());
        for (auto& o : tmp) o.near_ties = 0;
        PT_CUDA(cudaMemcpyAsync(c->d_obs, tmp.data(), (size_t)c->R() * sizeof(pt_obs), cudaMemcpyHostToDevice, c->stream));
        PT_CUDA(cudaStreamSynchronize(c->stream));   // tmp goes out of scope
    }
    c->sweep = sweep;
    return pt_sync(c);
}

int pt_get_couplings(pt_ctx* c, int32_t* Jq) {
    if (!c || !Jq) return fail(PT_EINVAL, "NULL argument");
    DeviceGuard guard(c->device);
    PT_CUDA(cudaMemcpy(Jq, c->d_Jq, (size_t)c->L * sizeof(int32_t), cudaMemcpyDeviceToHost));
    return PT_OK;
}

int64_t pt_sweep_counter(pt_ctx* c) { return c ? c->sweep : -1; }

int pt_create_shard(pt_ctx** out, int L, int q, double sigma, int n_rep, const double* betas, uint64_t seed,
                    int ens_base, int rep_base, int n_local) {
    if (out) *out = nullptr;
    if (rep_base < 0 || n_local < 1 || n_rep < 1 || (long long)rep_base + n_local > n_rep)
        return fail(PT_EINVAL, "need 0 <= rep_base, n_local >= 1 and rep_base + n_local <= n_rep");
    pt_ctx* c = nullptr;
    int rc = pt_create_ex(&c, L, q, sigma, 1, n_rep, betas, seed, ens_base);
    if (rc) return rc;
    if (c->variant != PT_VARIANT_DIRECT) {
        pt_destroy(c);
        return fail(PT_EINVAL, "slot-sharded contexts need the direct variant (L % 64 == 0, 64 <= L <= 10240)");
    }
    c->rep_base = rep_base;
    c->n_local = n_local;
    *out = c;
    return PT_OK;
}

int pt_energy_storage_dev_async(pt_ctx* c, int64_t* E_out_dev) {
    if (!c || !E_out_dev) return fail(PT_EINVAL, "NULL argument");
    DeviceGuard guard(c->device);
    const int n = c->n_local ? c->n_local : c->R();
    PT_CUDA(cudaMemcpyAsync(E_out_dev, c->d_E + c->rep_base, (size_t)n * sizeof(long long), cudaMemcpyDeviceToDevice,
                            c->stream));
    return PT_OK;
}

int pt_energy_storage_dev(pt_ctx* c, int64_t* E_out_dev) {
    int rc = pt_energy_storage_dev_async(c, E_out_dev);
    return rc ? rc : pt_sync(c);
}

int pt_swap_external_async(pt_ctx* c, const int64_t* E_all_dev) {
    if (!c || !E_all_dev) return fail(PT_EINVAL, "NULL argument");
    if (!c->n_local) return fail(PT_EINVAL, "pt_swap_external is for slot-sharded contexts (pt_create_shard)");
    DeviceGuard guard(c->device);
    PT_CUDA(cudaMemcpyAsync(c->d_E, E_all_dev, (size_t)c->n_rep * sizeof(long long), cudaMemcpyDeviceToDevice,
                            c->stream));
    ptk::swap_kernel<<<1, 256, 0, c->stream>>>(c->dev(), (uint32_t)c->sweep);
    PT_CUDA(cudaGetLastError());
    return PT_OK;
}

int pt_swap_external(pt_ctx* c, const int64_t* E_all_dev) {
    int rc = pt_swap_external_async(c, E_all_dev);
    return rc ? rc : pt_sync(c);
}

int pt_get_perm(pt_ctx* c, int32_t* perm) {
    if (!c || !perm) return fail(PT_EINVAL, "NULL argument");
    DeviceGuard guard(c->device);
    int rc = pt_sync(c);
    if (rc) return rc;
    PT_CUDA(cudaMemcpy(perm, c->d_perm, (size_t)c->R() * sizeof(int), cudaMemcpyDeviceToHost));
    return PT_OK;
}

#ifdef PT_TIMING
// Development builds only (-DPT_TIMING): per-warp clock sums of the sweep kernel, [R][32][8].
int pt_debug_timing(pt_ctx* c, long long* out) {
    if (!c || !out || !c->d_dbg) return fail(PT_EINVAL, "no timing buffer");
    PT_CUDA(cudaMemcpy(out, c->d_dbg, (size_t)c->R() * 32 * 8 * sizeof(long long), cudaMemcpyDeviceToHost));
    PT_CUDA(cudaMemset(c->d_dbg, 0, (size_t)c->R() * 32 * 8 * sizeof(long long)));
    return PT_OK;
}
#endif

int pt_measure_peaks(double* rates, int n) {
    if (!rates || n < PT_PEAK_PATTERNS * 4) return fail(PT_EINVAL, "rates must hold PT_PEAK_PATTERNS * 4 doubles");
    int dev = 0, n_sm = 0;
    PT_CUDA(cudaGetDevice(&dev));
    PT_CUDA(cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev));
    long long* d_clk = nullptr;
    uint32_t* d_sink = nullptr;
    PT_CUDA(cudaMalloc(&d_clk, (size_t)n_sm * sizeof(long long)));
    cudaError_t err = cudaMalloc(&d_sink, sizeof(uint32_t));
    if (err != cudaSuccess) { cudaFree(d_clk); return fail(PT_ENOMEM, cudaGetErrorString(err)); }
    std::vector<long long> clk(n_sm);
    int rc = PT_OK;
    for (int p = 0; p < PT_PEAK_PATTERNS && rc == PT_OK; ++p) {
        ptk::peak_kernel_t k = ptk::peak_kernel_of(p);
        for (int w = 1; w <= 4 && rc == PT_OK; ++w) {
            const int threads = 128 * w;   // w warps on each of the 4 sub-partitions
            for (int rep = 0; rep < 2; ++rep) k<<<n_sm, threads>>>(d_clk, d_sink, 12345u + rep);   // first run warms up
            err = cudaMemcpy(clk.data(), d_clk, (size_t)n_sm * sizeof(long long), cudaMemcpyDeviceToHost);
            if (err != cudaSuccess) { rc = fail(PT_ECUDA, cudaGetErrorString(err)); break; }
            std::sort(clk.begin(), clk.end());
            const double med = (double)clk[n_sm / 2];
            // lane-operations (bytes for the LDS pattern) per clock and SM
            const double per_thread = ptk::peak_counted_ops(p);
            rates[p * 4 + (w - 1)] = p == ptk::PEAK_LDS128 ? per_thread * threads / med : per_thread * threads / med;
        }
    }
    cudaFree(d_clk);
    cudaFree(d_sink);
    return rc;
}

int pt_set_variant(pt_ctx* c, int variant) {
    if (!c) return fail(PT_EINVAL, "ctx is NULL");
    if (c->n_local && variant == PT_VARIANT_FIELD) return fail(PT_EINVAL, "slot-sharded contexts need the direct variant");
    if (c->site_order == PT_ORDER_RANDOM && variant != PT_VARIANT_FIELD)
        return fail(PT_EINVAL, "random site order runs in the field variant only");
    const bool to_float = variant == PT_VARIANT_FP32 || variant == PT_VARIANT_FP64;
    if (c->n_local && to_float) return fail(PT_EINVAL, "slot-sharded contexts need the direct variant");
    DeviceGuard guard(c->device);
    int v = 0;
    int rc = resolve_variant(c->L, c->q, c->rowsum, variant, &v);
    if (rc) return rc;
    const bool from_float = c->variant == PT_VARIANT_FP32 || c->variant == PT_VARIANT_FP64;
    if (from_float && v != c->variant) {
        // the floating-point running energies carry rounding errors: the exact variants restart from the recount
        // (a change between fp32 and fp64 re-enters from the exact energies as well)
        c->ef_valid = false;
        rc = recompute_energy(c, c->d_E);
        if (rc) return rc;
    }
    c->variant = v;
    return PT_OK;
}

int pt_get_variant(pt_ctx* c) { return c ? c->variant : PT_EINVAL; }

int pt_describe(pt_ctx* c, char* out, int n) {
    if (!c || !out || n < 1) return fail(PT_EINVAL, "ctx or out is NULL, or n < 1");
    DeviceGuard guard(c->device);
    char line[256];
    if (c->variant == PT_VARIANT_DIRECT) {
        if (!c->direct_kern) c->direct_kern = ptk::select_direct_kernel(c->dev(), c->r_hi, c->device, &c->coresident);
        cudaFuncAttributes fa;
        PT_CUDA(cudaFuncGetAttributes(&fa, (const void*)c->direct_kern));
        const int cw = ptk::direct_chain_warps_of(c->direct_kern);
        // near quads per thread of the build in use: find the (build, wide) combination that gives this kernel
        int nq = -1;
        const ptk::Dev d = c->dev();
        for (int minb : {1, 4, 2})
            for (int wide4 = 1; wide4 >= 0 && nq < 0; --wide4)
                if (c->direct_kern == ptk::direct_kernel_variant(d, c->r_hi, minb, wide4 != 0))
                    nq = ptk::direct_effective_nearq(d, c->r_hi, minb, wide4 != 0);
        if (nq < 0) nq = 0;
        snprintf(line, sizeof line,
                 "direct: threads=%d regs=%d resident_ctas=%d near_window=%d near_quads=%d chain_warps=%d persistent=%d",
                 ptk::direct_threads(c->L, cw), fa.numRegs, c->coresident, nq ? ptk::direct_near_off(c->r_hi) : 0, nq, cw,
                 persistent_ok(c) ? 1 : 0);
    } else if (c->variant == PT_VARIANT_FIELD) {
        const int C = field_cluster_of(c);
        const size_t smem = C ? ptk::field_cluster_smem_bytes(c->L, c->q, C)
                              : ptk::field_smem_bytes(c->L, c->q, c->site_order == PT_ORDER_RANDOM);
        snprintf(line, sizeof line, "field: cluster=%d threads=%d smem=%zu", C, ptk::FIELD_THREADS, smem);
    } else {
        snprintf(line, sizeof line, "%s: threads=%d", c->variant == PT_VARIANT_FP32 ? "fp32" : "fp64", ptk::FLOAT_THREADS);
    }
    snprintf(out, (size_t)n, "%s", line);
    return PT_OK;
}

int pt_set_site_order(pt_ctx* c, int order) {
    if (!c) return fail(PT_EINVAL, "ctx is NULL");
    if (order != PT_ORDER_SEQUENTIAL && order != PT_ORDER_RANDOM) return fail(PT_EINVAL, "unknown site order");
    if (order == PT_ORDER_RANDOM) {
        if (c->n_local) return fail(PT_EINVAL, "slot-sharded contexts sweep in sequential order");
        if (ptk::field_smem_bytes(c->L, c->q, true) + 256 > kSmemLimit)
            return fail(PT_ECAPACITY, "local-field table and step lists do not fit in shared memory");
        int rc = pt_set_variant(c, PT_VARIANT_FIELD);   // (leaving a floating-point variant recounts the energies)
        if (rc) return rc;
    }
    c->site_order = order;
    return PT_OK;
}

int pt_set_stream(pt_ctx* c, void* cuda_stream) {
    if (!c) return fail(PT_EINVAL, "ctx is NULL");
    DeviceGuard guard(c->device);
    PT_CUDA(cudaStreamSynchronize(c->stream));
    c->stream = (cudaStream_t)cuda_stream;
    return PT_OK;
}

}  // extern "C"

// ---------------------------------------------------------------------------
// pt_energy_static (include/pt.h): total energies of caller-supplied configurations without any allocation.
// The scratch the recount needs -- the quantised coupling table Jq[L] (a1) and the packed spins -- lives in ONE
// file-scope device array that every GPU loading the library holds until exit.  In host code the array's NAME is a
// host-side stand-in, not a device address: its address on the current device is asked once per device with
// cudaGetSymbolAddress and that pointer is what the kernels get.  All calls share the array (it keeps the last call's
// contents; the flag word is cleared at the start of every call), so calls that overlap on the GPU race.
// ---------------------------------------------------------------------------
namespace {

constexpr int kStaticFlagWords = 64;                                    // word 0: a colour outside 1..q was seen
constexpr int kStaticSpinWords = PT_STATIC_MAX_SITES / 4;               // byte-wide packing (q > 16) is the widest
constexpr int kStaticWords = kStaticFlagWords + PT_STATIC_MAX_L + kStaticSpinWords;
static __device__ __align__(256) uint32_t g_static_scratch[kStaticWords];   // 1 114 368 bytes per GPU

constexpr int kMaxDevices = 64;
std::mutex g_static_mu;
uint32_t* g_static_ptr[kMaxDevices] = {};   // device address of g_static_scratch, by device ordinal

// One thread per packed word: API colours 1..q, one byte per site -> stored colours 0..q-1, `bits` bits per site.
__global__ void static_pack_kernel(const uint8_t* __restrict__ in, uint32_t* __restrict__ words, long long n_words,
                                   int bits, int q, uint32_t* __restrict__ flag) {
    const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (gid >= n_words) return;
    const int per = 32 / bits;
    const uint8_t* s = in + gid * per;
    uint32_t word = 0;
    bool bad = false;
    for (int n = 0; n < per; ++n) {
        const int v = s[n];
        bad |= v < 1 || v > q;
        word |= ((uint32_t)(v - 1) & ((1u << bits) - 1u)) << (bits * n);
    }
    words[gid] = word;
    if (bad) atomicOr(flag, 1u);
}

__global__ void static_status_kernel(const uint32_t* __restrict__ flag, int* __restrict__ status) {
    status[0] = (int)flag[0];
}

// Device address of the scratch array on the CURRENT device (asked once per device, with that device current).
int static_scratch(uint32_t** out) {
    int dev = 0;
    PT_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kMaxDevices) return fail(PT_EINVAL, "device ordinal beyond 63");
    std::lock_guard<std::mutex> lock(g_static_mu);
    if (!g_static_ptr[dev]) {
        uint32_t* p = nullptr;
        PT_CUDA(cudaGetSymbolAddress((void**)&p, g_static_scratch));
        g_static_ptr[dev] = p;
    }
    *out = g_static_ptr[dev];
    return PT_OK;
}

}  // namespace

extern "C" int pt_energy_static(int L, int q, double sigma, const uint8_t* spins_dev, int n_conf, int64_t* E_out_dev,
                                int* status_dev, void* cuda_stream) {
    if (L < 8 || (L % 8) != 0) return fail(PT_EINVAL, "L must be a multiple of 8, >= 8");
    if (L > PT_STATIC_MAX_L) return fail(PT_ECAPACITY, "pt_energy_static: L exceeds PT_STATIC_MAX_L (16384)");
    if (q < 2 || q > ptk::PT_QMAX) return fail(PT_EINVAL, "q must be in 2..64");
    if (!(sigma > 0.0) || !std::isfinite(sigma)) return fail(PT_EINVAL, "sigma must be finite and > 0");
    if (n_conf < 1) return fail(PT_EINVAL, "n_conf must be >= 1");
    if ((long long)n_conf * L > PT_STATIC_MAX_SITES)
        return fail(PT_ECAPACITY, "pt_energy_static: n_conf * L exceeds PT_STATIC_MAX_SITES (1048576); split the call");
    if (!spins_dev || !E_out_dev) return fail(PT_EINVAL, "spins_dev and E_out_dev must not be NULL");
    uint32_t* scratch = nullptr;
    int rc = static_scratch(&scratch);
    if (rc) return rc;
    cudaStream_t stream = (cudaStream_t)cuda_stream;
    uint32_t* flag = scratch;
    int32_t* Jq = (int32_t*)(scratch + kStaticFlagWords);
    uint32_t* words = scratch + kStaticFlagWords + PT_STATIC_MAX_L;

    ptk::Dev d = {};
    d.L = L; d.q = q; d.n_ens = 1; d.n_rep = n_conf; d.n_local = n_conf;
    d.bits = q <= 16 ? 4 : 8;
    d.W = L * d.bits / 32;
    d.Jq = Jq; d.spins = words;
    const long long n_words = (long long)n_conf * d.W;

    PT_CUDA(cudaMemsetAsync(flag, 0, kStaticFlagWords * sizeof(uint32_t), stream));   // the array keeps the last call's contents
    ptk::jstar_kernel<<<(L / 2 + 128) / 128, 128, 0, stream>>>(L, sigma, Jq, nullptr);          // a1: all of Jq[0..L-1]
    PT_CUDA(cudaGetLastError());
    static_pack_kernel<<<(unsigned)((n_words + 255) / 256), 256, 0, stream>>>(spins_dev, words, n_words, d.bits, q, flag);
    PT_CUDA(cudaGetLastError());
    const size_t smem = (size_t)(L + d.W) * 4;
    if (smem > 48 * 1024) PT_CUDA((cudaError_t)ptk::allow_max_dynamic_smem((const void*)ptk::energy_kernel, 1024));
    ptk::energy_kernel<<<n_conf, 256, smem, stream>>>(d, (long long*)E_out_dev);                // a6
    PT_CUDA(cudaGetLastError());
    if (status_dev) {
        static_status_kernel<<<1, 1, 0, stream>>>(flag, status_dev);
        PT_CUDA(cudaGetLastError());
    }
    return PT_OK;
}

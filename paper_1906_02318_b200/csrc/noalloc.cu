// noalloc.cu -- mpmi_tick_noalloc (include/mpmi.h): one whole MPMI-SC tick (Algorithm 2) for callers that
// cannot allocate -- no context, no cudaMalloc / cudaFree / cudaHostAlloc, no graph, no stream or event creation.
//
// The tick kernel is the shared-memory-model instantiation of rollout_reg_kernel (rollout_reg.cuh, KC = false, two candidates
// per thread): a1 sample, a2 lift, a3 + a4 rollout with the per-step safe test, a5 key, a6 + a7 cross-CTA argmin and result.
// Where a context keeps that kernel's two pieces of device scratch in cudaMalloc memory (mpmi_api.cu: d_KTa, the model in the
// kernel's own layout; d_state, the cross-CTA selection state), this entry keeps them in ONE file-scope __device__ array:
//
//     g_noalloc_scratch  [0, 256)       TickState: best key, counters, arrival ticket of the CTAs (block_select_and_finalise)
//                        [256, 4864)    KTa, the augmented transposed model (D + M) x D of the caller's K and B, physical dims
//                                       in the internal order (constrained dims first), zero padded to D = 8 / 16 / 32
//
// 8 KB per GPU that loads the library, held until the process exits.  That fixes the maximum: d <= 32 (padded D <= 32, m <= 4);
// anything larger is rejected with MPMI_ERR_UNSUPPORTED and a message (mpmi_noalloc_last_error).  Every call re-packs the model
// and re-arms the selection state in a one-CTA kernel ahead of the tick kernel, so nothing is assumed about what the last call
// left behind.  All calls on a GPU share the array: two calls whose kernels overlap on the GPU (different streams, or two host
// threads) race on it -- the caller serialises them.
//
// In host code `g_noalloc_scratch` is a host-side stand-in of the symbol, not a device address; the address the kernels get
// comes from cudaGetSymbolAddress, taken once per device with that device current (scratch_of below).
#include <cmath>
#include <cstring>
#include <mutex>
#include <string>
#include <cuda_runtime.h>
#include "../../include/mpmi.h"
#include "rollout_reg.cuh"

using namespace mpmi;

namespace {

constexpr int kNoallocMaxD = 32;
constexpr int kNoallocStateBytes = 256;
constexpr int kNoallocScratchBytes = 8192;
static_assert(sizeof(TickState) <= kNoallocStateBytes, "selection state must fit its slot");
static_assert(kNoallocStateBytes + (kNoallocMaxD + MPMI_MAX_M) * kNoallocMaxD * (int)sizeof(float) <= kNoallocScratchBytes, "scratch too small");

static __device__ __align__(256) unsigned char g_noalloc_scratch[kNoallocScratchBytes];

// Packs the caller's K (d x d, row-major) and B (d x m) into KTa[c][r] (c < D: K[r][c]; c >= D: B[r][c - D]; internal order of
// the physical dims, zero padding) -- what mpmi_create does on the host -- and re-arms the selection state.
__global__ void __launch_bounds__(256) noalloc_pack_kernel(const __grid_constant__ DevCfg cfg, const float *K, const float *B,
                                                           TickState *st, float *kta) {
    const int D = cfg.D, d = cfg.d, n = cfg.n, m = cfg.m;
    for (int i = threadIdx.x; i < (D + m) * D; i += blockDim.x) {
        const int c = i / D, r = i - c * D;
        float v = 0.f;
        if (r < d) {
            const int ro = r < n ? cfg.perm[r] : r;
            if (c < D) {
                if (c < d) v = K[(size_t)ro * d + (c < n ? cfg.perm[c] : c)];
            } else {
                v = B[(size_t)ro * m + (c - D)];
            }
        }
        kta[i] = v;
    }
    if (threadIdx.x == 0) {
        st->best_key = kKeyNone; st->n_exec = 0ull; st->n_safe = 0u; st->ticket = 0u; st->work = 0u; st->pad = 0u;
    }
}

template <int D>
KernFn pick_m(int M) {
    switch (M) {
        case 1: return rollout_reg_kernel<D, 1, 1, MODE_TICK, false, false>;
        case 2: return rollout_reg_kernel<D, 2, 1, MODE_TICK, false, false>;
        case 3: return rollout_reg_kernel<D, 3, 1, MODE_TICK, false, false>;
        case 4: return rollout_reg_kernel<D, 4, 1, MODE_TICK, false, false>;
    }
    return nullptr;
}
KernFn pick_tick(int D, int M) { return D == 8 ? pick_m<8>(M) : D == 16 ? pick_m<16>(M) : D == 32 ? pick_m<32>(M) : nullptr; }

thread_local std::string g_err;
int fail(int code, const std::string &msg) { g_err = "mpmi_tick_noalloc: " + msg; return code; }

// device address of the scratch array, once per device, with that device current
constexpr int kMaxDevices = 64;
std::mutex g_mu;
unsigned char *g_scratch_ptr[kMaxDevices] = {};
int g_cc_major[kMaxDevices] = {};

int scratch_of(int dev, unsigned char **out) {
    std::lock_guard<std::mutex> lk(g_mu);
    if (!g_scratch_ptr[dev]) {
        int major = 0;
        cudaError_t e = cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev);
        if (e != cudaSuccess) return fail(MPMI_ERR_CUDA, std::string("cudaDeviceGetAttribute: ") + cudaGetErrorString(e));
        g_cc_major[dev] = major;
        if (major != 10) return fail(MPMI_ERR_UNSUPPORTED, "device is not compute capability 10.x (kernels are sm_100a only)");
        void *p = nullptr;
        e = cudaGetSymbolAddress(&p, g_noalloc_scratch);
        if (e != cudaSuccess) return fail(MPMI_ERR_CUDA, std::string("cudaGetSymbolAddress: ") + cudaGetErrorString(e));
        g_scratch_ptr[dev] = static_cast<unsigned char *>(p);
    }
    *out = g_scratch_ptr[dev];
    return MPMI_OK;
}

bool finite_all(const float *p, int n) {
    for (int i = 0; i < n; i++) if (!std::isfinite(p[i])) return false;
    return true;
}

}  // namespace

extern "C" {

const char *mpmi_noalloc_last_error(void) { return g_err.c_str(); }

int mpmi_tick_noalloc(const mpmi_config *cfg, const float *d_x0, const float *d_u_user, uint64_t tick, void *cuda_stream,
                      mpmi_result *d_out) {
    g_err.clear();
    if (!cfg || !d_x0 || !d_u_user || !d_out) return fail(MPMI_ERR_INVALID, "null config, input or output pointer");
    const int n = cfg->n, m = cfg->m, d = cfg->d;
    if (n <= 0 || m <= 0 || d <= 0 || cfg->N <= 0 || cfg->H <= 0) return fail(MPMI_ERR_INVALID, "n, m, d, N, H must be positive");
    if (d > kNoallocMaxD)
        return fail(MPMI_ERR_UNSUPPORTED, "d = " + std::to_string(d) + " exceeds the maximum of 32: the static scratch array holds a (32 + 4) x 32 model "
                                          "(use mpmi_create / mpmi_step_device for larger lifted dims)");
    if (m > MPMI_MAX_M || n > MPMI_MAX_N) return fail(MPMI_ERR_UNSUPPORTED, "m > 4 or n > 16");
    if (n > d) return fail(MPMI_ERR_INVALID, "n > d: the first n lifted features must be the state");
    if (cfg->N > MPMI_MAX_CAND || cfg->H > 65535) return fail(MPMI_ERR_UNSUPPORTED, "N or H too large");
    if (!cfg->K || !cfg->B || !cfg->u_lo || !cfg->u_hi) return fail(MPMI_ERR_INVALID, "null K, B, u_lo or u_hi");
    if (!finite_all(cfg->u_lo, m) || !finite_all(cfg->u_hi, m)) return fail(MPMI_ERR_INVALID, "non-finite input box");
    for (int j = 0; j < m; j++) if (cfg->u_lo[j] > cfg->u_hi[j]) return fail(MPMI_ERR_INVALID, "u_lo > u_hi");
    if (cfg->noise_sigma != 0.f) return fail(MPMI_ERR_UNSUPPORTED, "prediction noise is not built into this entry point (noise_sigma must be 0)");
    if (cfg->model != MPMI_MODEL_LINEAR) return fail(MPMI_ERR_UNSUPPORTED, "linear lifted model only");
    if (cfg->sampler != MPMI_SAMPLER_PHILOX && cfg->sampler != MPMI_SAMPLER_GRID) return fail(MPMI_ERR_INVALID, "unknown sampler");
    if (cfg->sampler == MPMI_SAMPLER_GRID) {
        if (!cfg->grid_counts) return fail(MPMI_ERR_INVALID, "grid sampler without grid_counts");
        long long prod = 1;
        for (int j = 0; j < m; j++) {
            if (cfg->grid_counts[j] <= 0) return fail(MPMI_ERR_INVALID, "grid count <= 0");
            prod *= cfg->grid_counts[j];
            if (prod > MPMI_MAX_CAND) break;
        }
        if (prod != cfg->N) return fail(MPMI_ERR_INVALID, "N != product of grid_counts");
    }
    const mpmi_lift_spec &L = cfg->lift;
    if (L.kind == MPMI_LIFT_MONO) {
        if (!L.terms) return fail(MPMI_ERR_INVALID, "MONO lift without terms");
    } else if (L.kind == MPMI_LIFT_RFF) {
        if (d > n && (!L.W || !L.b)) return fail(MPMI_ERR_INVALID, "RFF lift without W or b");
        if (!std::isfinite(L.scale)) return fail(MPMI_ERR_INVALID, "non-finite RFF scale");
    } else {
        return fail(MPMI_ERR_INVALID, "unknown lift kind");
    }
    const mpmi_safe_spec &S = cfg->safe;
    if (S.nbounds < 0 || S.nbounds > MPMI_MAX_BOUNDS || (S.nbounds > 0 && (!S.idx || !S.lo || !S.hi))) return fail(MPMI_ERR_INVALID, "bad box constraints");
    for (int q = 0; q < S.nbounds; q++) {
        if (S.idx[q] < 0 || S.idx[q] >= n) return fail(MPMI_ERR_INVALID, "box constraint index >= n");
        if (std::isnan(S.lo[q]) || std::isnan(S.hi[q])) return fail(MPMI_ERR_INVALID, "NaN box limit");
    }
    if (!std::isfinite(S.inflate)) return fail(MPMI_ERR_INVALID, "non-finite inflate");
    if (S.annulus) {
        if (S.ix < 0 || S.ix >= n || S.iy < 0 || S.iy >= n || S.ix == S.iy) return fail(MPMI_ERR_INVALID, "bad annulus coordinates");
        if (!std::isfinite(S.cx) || !std::isfinite(S.cy) || !std::isfinite(S.rmin) || !std::isfinite(S.rmax) || S.rmin < 0)
            return fail(MPMI_ERR_INVALID, "bad annulus radii");
    }
    const long long ncg = (long long)cfg->N + (cfg->include_user ? 1 : 0);
    if (!((cfg->shard_begin == 0 && cfg->shard_count == 0) || (cfg->shard_begin == 0 && cfg->shard_count == ncg)))
        return fail(MPMI_ERR_UNSUPPORTED, "the whole candidate set only (no shards)");

    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return fail(MPMI_ERR_CUDA, std::string("cudaGetDevice: ") + cudaGetErrorString(e));
    if (cfg->device >= 0 && cfg->device != dev) return fail(MPMI_ERR_INVALID, "cfg->device is not the current device (this entry point never switches devices)");
    if (dev < 0 || dev >= kMaxDevices) return fail(MPMI_ERR_UNSUPPORTED, "device ordinal >= 64");
    unsigned char *scratch = nullptr;
    const int rc = scratch_of(dev, &scratch);
    if (rc != MPMI_OK) return rc;

    // ---- the kernels' configuration, by value (same folding of the safe set and internal order as mpmi_create)
    DevCfg dc;
    std::memset(&dc, 0, sizeof dc);
    int perm[MPMI_MAX_N], np = 0;
    bool used[MPMI_MAX_N] = {};
    if (S.annulus) { perm[np++] = S.ix; perm[np++] = S.iy; used[S.ix] = used[S.iy] = true; }
    for (int j = 0; j < n; j++) {
        bool boxed = false;
        for (int q = 0; q < S.nbounds; q++) boxed = boxed || S.idx[q] == j;
        if (boxed && !used[j]) { perm[np++] = j; used[j] = true; }
    }
    for (int j = 0; j < n; j++) if (!used[j]) perm[np++] = j;
    const int D = d <= 8 ? 8 : d <= 16 ? 16 : 32;
    dc.n = n; dc.m = m; dc.d = d; dc.D = D;
    dc.N = cfg->N; dc.H = cfg->H; dc.include_user = cfg->include_user ? 1 : 0;
    dc.ncand_global = ncg; dc.shard_begin = 0; dc.shard_count = ncg;
    dc.sampler = cfg->sampler;
    dc.seed_lo = (unsigned)cfg->seed; dc.seed_hi = (unsigned)(cfg->seed >> 32);
    for (int j = 0; j < kMaxM; j++) {
        dc.grid_counts[j] = (cfg->sampler == MPMI_SAMPLER_GRID && j < m) ? cfg->grid_counts[j] : 1;
        dc.u_lo[j] = j < m ? cfg->u_lo[j] : 0.f;
        dc.u_hi[j] = j < m ? cfg->u_hi[j] : 0.f;
    }
    dc.lift_kind = L.kind; dc.rff_scale = L.scale;
    for (int j = 0; j < kMaxN; j++) { dc.blo[j] = -INFINITY; dc.bhi[j] = INFINITY; dc.perm[j] = (unsigned char)(j < n ? perm[j] : j); }
    for (int q = 0; q < S.nbounds; q++) {
        int ji = 0;
        while (perm[ji] != S.idx[q]) ji++;
        const float lo = (float)((double)S.lo[q] + (double)S.inflate), hi = (float)((double)S.hi[q] - (double)S.inflate);
        dc.blo[ji] = std::fmax(dc.blo[ji], lo);
        dc.bhi[ji] = std::fmin(dc.bhi[ji], hi);
        dc.bmask |= 1u << ji;
    }
    dc.annulus = S.annulus ? 1 : 0;
    if (S.annulus) {
        const double rmin = (double)S.rmin + S.inflate, rmax = (double)S.rmax - S.inflate;
        dc.cx = S.cx; dc.cy = S.cy;
        dc.rmin2 = (float)(rmin * rmin); dc.rmax2 = rmax < 0 ? -1.f : (float)(rmax * rmax);
    }
    dc.noise_sigma = 0.f; dc.model = MPMI_MODEL_LINEAR;
    TickState *st = reinterpret_cast<TickState *>(scratch);
    float *kta = reinterpret_cast<float *>(scratch + kNoallocStateBytes);
    dc.KTa = kta;
    dc.terms = L.kind == MPMI_LIFT_MONO ? L.terms : nullptr;       // DEVICE pointers here (header): features >= n keep their place in the internal order
    dc.W = L.W; dc.b = L.b;

    const KernFn fn = pick_tick(D, m);
    if (!fn) return fail(MPMI_ERR_UNSUPPORTED, "no kernel for this (d, m)");
    cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
    {
        const float *K = cfg->K, *B = cfg->B;
        void *args[5] = {(void *)&dc, (void *)&K, (void *)&B, (void *)&st, (void *)&kta};
        e = cudaLaunchKernel((const void *)noalloc_pack_kernel, dim3(1), dim3(256), args, 0, s);
        if (e != cudaSuccess) return fail(MPMI_ERR_CUDA, std::string("launch of the pack kernel: ") + cudaGetErrorString(e));
    }
    KArgs a{};
    a.x0 = d_x0; a.u_user = d_u_user; a.tick_val = tick; a.st = st; a.out = d_out; a.kslot = 0;
    const long long cpb = 2LL * kRegBlock;                          // P = 1: two candidates per thread
    const long long blocks = (ncg + cpb - 1) / cpb;
    void *args[2] = {(void *)&dc, (void *)&a};
    e = cudaLaunchKernel((const void *)fn, dim3((unsigned)blocks), dim3(kRegBlock), args, 0, s);
    if (e != cudaSuccess) return fail(MPMI_ERR_CUDA, std::string("launch of the tick kernel: ") + cudaGetErrorString(e));
    return MPMI_OK;
}

}  // extern "C"

// mpmi_api.cu -- host runtime and C ABI (include/mpmi.h) of the B200-native MPMI-SC tick.
// Context creation (validation, internal re-ordering / padding of the model, upload), kernel
// choice, the per-tick CUDA graph (param H2D -> fused tick kernel -> result D2H),
// pinned staging, and the benchmark entry mpmi_rollout_batch.  No CPU fallback: every step of the
// path runs in the kernels of rollout_reg.cuh / rollout_tile.cuh.
#include <atomic>
#include <chrono>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>
#include <string>
#include <thread>
#include <vector>
#if defined(__x86_64__) || defined(__i386__)
#include <immintrin.h>
#endif
#include <cuda_runtime.h>
#include "../../include/mpmi.h"
#include "mpmi_device.cuh"
#include "kernel_args.cuh"
#include "binning.cuh"
#include "bound.cuh"
#include "rollout_split.cuh"

using namespace mpmi;


struct HostBlock { mpmi_result r; int deferred; int pad[3]; };      // mapped pinned memory the finalising CTA writes

struct mpmi_ctx {
    DevCfg dc;
    int kslot = -1;                                   // constant-memory slot of the model (register kernels), -1 = none
    int device = 0, sm_count = 0;
    int variant = 0, P = 1, smem = 0, regs = 0;
    int block = 128, cand_per_block = 0;              // launch geometry of the tick kernel
    int bblock = 128, bcand_per_block = 0;            // launch geometry of the batch kernel
    KernFn k_tick = nullptr, k_batch = nullptr;
    int bsmem = 0;                                    // dynamic shared memory of the batch kernel
    bool bpersistent = false;                         // batch kernel is a persistent one-CTA-per-SM kernel
    // affine-in-u fast path (rollout_affine.cuh)
    bool affine = false;
    KernFn k_base = nullptr, k_batch_aff = nullptr;
    // trajectory dumps (a9) at D <= 32 use the 2-candidates-per-thread packing: fewer registers, more resident CTAs,
    // and the HBM stores overlap the FMAs better (measured 5.0 -> 5.9 TB/s at d = 16, 5.6 -> 6.7 TB/s at d = 8)
    KernFn k_batch_dump = nullptr;
    float *d_affA = nullptr, *d_affG = nullptr;
    cudaGraphNode_t n_base = nullptr;
    float *d_KTa = nullptr, *d_W = nullptr, *d_b = nullptr, *d_affM = nullptr;
    uint8_t *d_terms = nullptr;
    TickState *d_state = nullptr;
    mpmi_result *h_res = nullptr, *d_res_mapped = nullptr;   // pinned + mapped: the tick kernel writes the result here
    // the tick as ONE CUDA graph: [cell histogram, scatter,] fused tick kernel.  The tick inputs travel
    // inside the kernel-node parameters (updated per launch), the result comes back through mapped memory.
    cudaGraph_t graph = nullptr;
    cudaGraphExec_t exec = nullptr;
    cudaGraphNode_t n_hist = nullptr, n_scatter = nullptr, n_tick = nullptr;
    unsigned bin_grid = 0, tick_grid = 0;
    KArgs ga{};
    BinArgs gb{};
    unsigned seq = 0;
    cudaStream_t pending_stream = nullptr;
    bool pending = false;
    // spatial binning of Philox candidates (binning.cuh)
    bool binning = false;
    BinArgs bin{};
    int *d_hist = nullptr, *d_cursor = nullptr, *d_perm = nullptr;
    unsigned *d_bin_ticket = nullptr;
    // life-time order (binning.cuh): predicted steps of the local sampled candidates from the affine form
    bool predict = false;
    int *d_pred = nullptr;
    const void *k_pred = nullptr;    // bin_predict_kernel<aff_np>
    int tc_ctas = 1;                 // persistent CTAs per SM (4 for the tensor-core kernel at D = 32)
    long long lat_cap = 0;           // latency kernel: CTAs resident at once (its grid never exceeds them: rollout_lat.cuh)
    // verified tensor-core tick: the tcgen05 kernel defers the candidates that came within tau_i(k) (bound.cuh) of the
    // safe-set boundary to the FP32 kernel (register kernel at D = 32, warp-tile kernel at D = 128), which merges them and
    // finalises (kernel_args.cuh: recheck).  tau comes per tick from bound_err_kernel -> bound_tau_kernel.
    KernFn k_recheck = nullptr, k_batch_recheck = nullptr, k_batch_fp32 = nullptr;
    int *d_recheck = nullptr;
    unsigned *d_recheck_count = nullptr;
    unsigned recheck_grid = 0;
    int recheck_block = kRegBlock, recheck_smem = 0, fp32_smem = 0;
    bool recheck_persistent = false;
    int rc_warps = 0;                // MPMI_RC_WARPS (measurement): active warps per CTA of the d = 128 second pass
    float recheck_tau_scale = 1.f;   // MPMI_TC_TAU_SCALE (measures how conservative the bound is; not a tuning knob)
    cudaGraphNode_t n_recheck = nullptr, n_berr = nullptr, n_btau = nullptr;
    const void *k_berr = nullptr, *k_btau = nullptr;
    unsigned berr_block = 64;
    float *d_bnd_kpow = nullptr, *d_bnd_mid = nullptr, *d_bnd_econst = nullptr, *d_bnd_w = nullptr, *d_bnd_e = nullptr, *d_bnd_tau = nullptr;
    cudaStream_t side = nullptr;     // plain-launch entries: the bound kernels run beside the binning kernels
    cudaEvent_t ev_fork = nullptr, ev_join = nullptr;
    int *d_deferred_mapped = nullptr;
    KArgs gr{};
    // mpmi_profile_enable: CUDA events around the tick kernel and the second pass of the plain-launch entries (ring of kProfRing ticks)
    unsigned long long *timeline = nullptr;   // mpmi_profile_timeline: caller's device buffer, or null
    bool prof = false;
    std::vector<cudaEvent_t> prof_ev;     // 3 per slot: before the tick kernel, after it, after the second pass
    unsigned prof_n = 0;
    std::string err;
};

namespace mpmi {
// a7 for the sharded path: reduce G partials and decode.
__global__ void shard_finalise_kernel(const __grid_constant__ DevCfg cfg, const mpmi_partial *parts, int G,
                                      const float *u_user, unsigned long long tick, mpmi_result *out) {
    if (threadIdx.x != 0 || blockIdx.x != 0) return;
    unsigned long long k = kKeyNone, ne = 0; unsigned ns = 0;
    for (int g = 0; g < G; g++) {
        k = parts[g].key < k ? parts[g].key : k;
        ns += (unsigned)parts[g].n_safe; ne += (unsigned long long)parts[g].n_exec;
    }
    float u_h[kMaxM];
    clamp_user(cfg, u_user, u_h);
    decode_result(cfg, k, ne, ns, tick, u_h, out);
}

}  // namespace mpmi

namespace {

constexpr unsigned kProfRing = 64;
constexpr long long kLatMaxCand = 24576;        // <= this many candidates: latency kernel (measured: 125 vs 155 us at 2^14, 210 vs 164 us at 2^15)
// D = 32: the verified tensor-core tick takes over where the register kernel needs a second CTA on an SM (256 candidates per CTA: its tick
// then doubles, 157 -> 273 us on 148 SMs; the tensor-core tick without binning: 177 us at 40,000 candidates, 193 us at 2^16); its binning
// pays from ~80,000 candidates (2^16: 193 us without, 204 us with; 98,304: 256 / 234 us)
constexpr long long kTc32CandPerCta = 256, kTc32MinBinning = 81920;

thread_local std::string g_create_err;

inline void cpu_relax() {
#if defined(__x86_64__) || defined(__i386__)
    _mm_pause();
#elif defined(__aarch64__)
    asm volatile("yield" ::: "memory");
#endif
}

#define CU(ctx, call)                                                                      \
    do {                                                                                   \
        cudaError_t e_ = (call);                                                           \
        if (e_ != cudaSuccess) {                                                           \
            (ctx)->err = std::string(#call) + ": " + cudaGetErrorString(e_);               \
            return e_ == cudaErrorMemoryAllocation ? MPMI_ERR_NOMEM : MPMI_ERR_CUDA;       \
        }                                                                                  \
    } while (0)

int fail(mpmi_ctx *c, int code, const char *msg) {
    if (c) c->err = msg;
    g_create_err = msg;
    return code;
}

// kernel tables live in inst_reg.cu / inst_tile.cu, one translation unit per (D, MODE)
#define MPMI_DECL_REG(D) KernFn mpmi_pick_reg_##D##_tick(int M, int P, int kconst); KernFn mpmi_pick_reg_##D##_batch(int M, int P, int kconst); \
                         KernFn mpmi_pick_regn_##D##_tick(int M, int P, int kconst); KernFn mpmi_pick_regn_##D##_batch(int M, int P, int kconst); \
                         int mpmi_pick_reg_##D##_tick_setmodel(int, const float *, int); int mpmi_pick_reg_##D##_batch_setmodel(int, const float *, int); \
                         int mpmi_pick_regn_##D##_tick_setmodel(int, const float *, int); int mpmi_pick_regn_##D##_batch_setmodel(int, const float *, int);
#define MPMI_DECL_TILE(D) KernFn mpmi_pick_tile_##D##_tick(int M, int *smem); KernFn mpmi_pick_tile_##D##_batch(int M, int *smem); \
                          KernFn mpmi_pick_tilen_##D##_tick(int M, int *smem); KernFn mpmi_pick_tilen_##D##_batch(int M, int *smem);
}  // namespace
MPMI_DECL_REG(8) MPMI_DECL_REG(16) MPMI_DECL_REG(32) MPMI_DECL_TILE(64) MPMI_DECL_TILE(128)
KernFn mpmi_pick_tile_128_tick_rc(int M, int *smem); KernFn mpmi_pick_tile_128_batch_rc(int M, int *smem);
KernFn mpmi_pick_tilen_128_tick_rc(int M, int *smem); KernFn mpmi_pick_tilen_128_batch_rc(int M, int *smem);
KernFn mpmi_pick_reg_32_recheck(int M, int kconst); KernFn mpmi_pick_regn_32_recheck(int M, int kconst);
KernFn mpmi_pick_split_32(int M, int rs); KernFn mpmi_pick_splitn_32(int M, int rs);
KernFn mpmi_pick_relift(int n, int mode);
KernFn mpmi_pick_affine_base(int D); KernFn mpmi_pick_affine(int np, int mode);
KernFn mpmi_pick_tc_tick(int D, int *smem, int *threads, int *ctas_per_sm, int noise); KernFn mpmi_pick_tc_batch(int D, int *smem, int *threads, int *ctas_per_sm, int noise);
KernFn mpmi_pick_lat_8(int M, int R); KernFn mpmi_pick_lat_16(int M, int R); KernFn mpmi_pick_lat_32(int M, int R);
namespace {
KernFn pick_reg(int D, int M, int P, int mode, bool noise, int kconst = 1) {
    const bool t = mode == MODE_TICK;
    if (noise) {
        switch (D) {
            case 8: return t ? mpmi_pick_regn_8_tick(M, P, kconst) : mpmi_pick_regn_8_batch(M, P, kconst);
            case 16: return t ? mpmi_pick_regn_16_tick(M, P, kconst) : mpmi_pick_regn_16_batch(M, P, kconst);
            case 32: return t ? mpmi_pick_regn_32_tick(M, P, kconst) : mpmi_pick_regn_32_batch(M, P, kconst);
        }
        return nullptr;
    }
    switch (D) {
        case 8: return t ? mpmi_pick_reg_8_tick(M, P, kconst) : mpmi_pick_reg_8_batch(M, P, kconst);
        case 16: return t ? mpmi_pick_reg_16_tick(M, P, kconst) : mpmi_pick_reg_16_batch(M, P, kconst);
        case 32: return t ? mpmi_pick_reg_32_tick(M, P, kconst) : mpmi_pick_reg_32_batch(M, P, kconst);
    }
    return nullptr;
}
// constant-memory model slots of the register kernels: one per live context (kernel_args.cuh: kModelSlots)
// (__constant__ memory is per device, so is the slot table: 8 live register-kernel contexts per GPU)
constexpr int kMaxDevices = 64;
std::mutex g_slot_mu;
bool g_slot_used[kMaxDevices][kModelSlots] = {};
int slot_acquire(int dev) {
    if (dev < 0 || dev >= kMaxDevices) return -1;
    std::lock_guard<std::mutex> lk(g_slot_mu);
    for (int i = 0; i < kModelSlots; i++) if (!g_slot_used[dev][i]) { g_slot_used[dev][i] = true; return i; }
    return -1;
}
void slot_release(int dev, int i) {
    if (i < 0 || dev < 0 || dev >= kMaxDevices) return;
    std::lock_guard<std::mutex> lk(g_slot_mu);
    g_slot_used[dev][i] = false;
}
// the slot is filled in the translation units of the tick and batch kernels this context launches
int set_model(int D, bool noise, int slot, const float *kta, int nfloats) {
    int rc = 0;
#define MPMI_SET(D_) case D_: rc = noise ? (mpmi_pick_regn_##D_##_tick_setmodel(slot, kta, nfloats) | mpmi_pick_regn_##D_##_batch_setmodel(slot, kta, nfloats)) \
                                          : (mpmi_pick_reg_##D_##_tick_setmodel(slot, kta, nfloats) | mpmi_pick_reg_##D_##_batch_setmodel(slot, kta, nfloats)); break;
    switch (D) { MPMI_SET(8) MPMI_SET(16) MPMI_SET(32) default: rc = (int)cudaErrorInvalidValue; }
#undef MPMI_SET
    return rc;
}

KernFn pick_lat(int D, int M, int R) {
    return D == 8 ? mpmi_pick_lat_8(M, R) : D == 16 ? mpmi_pick_lat_16(M, R) : D == 32 ? mpmi_pick_lat_32(M, R) : nullptr;
}
KernFn pick_tile(int D, int M, int mode, int *smem, bool noise) {
    const bool t = mode == MODE_TICK;
    if (noise) {
        if (D == 64) return t ? mpmi_pick_tilen_64_tick(M, smem) : mpmi_pick_tilen_64_batch(M, smem);
        if (D == 128) return t ? mpmi_pick_tilen_128_tick(M, smem) : mpmi_pick_tilen_128_batch(M, smem);
        return nullptr;
    }
    if (D == 64) return t ? mpmi_pick_tile_64_tick(M, smem) : mpmi_pick_tile_64_batch(M, smem);
    if (D == 128) return t ? mpmi_pick_tile_128_tick(M, smem) : mpmi_pick_tile_128_batch(M, smem);
    return nullptr;
}

bool all_finite(const float *p, size_t n) {
    for (size_t i = 0; i < n; i++) if (!std::isfinite(p[i])) return false;
    return true;
}

// every launch returns its status: the callers hand it to CU() (no launch result is dropped)
cudaError_t launch_geom(const mpmi_ctx *c, KernFn fn, long long ncand, const KArgs &a0, cudaStream_t s, int cpb, int block, int smem,
                        bool persistent) {
    long long blocks = (ncand + cpb - 1) / cpb;
    if (blocks < 1) blocks = 1;
    if (fn == c->k_tick && c->variant == 3 && c->lat_cap > 0 && blocks > c->lat_cap) blocks = c->lat_cap;
    KArgs a = a0;
    if (persistent) {                            // persistent warp-tile / tensor-core kernel: one CTA per SM
        if (blocks > (long long)c->sm_count * c->tc_ctas) blocks = (long long)c->sm_count * c->tc_ctas;
        a.st = c->d_state; a.work = &c->d_state->work;
    }
    a.kslot = c->kslot;
    void *args[2] = {(void *)&c->dc, (void *)&a};
    return cudaLaunchKernel((const void *)fn, dim3((unsigned)blocks), dim3((unsigned)block), args, (size_t)smem, s);
}
cudaError_t launch(const mpmi_ctx *c, KernFn fn, long long ncand, const KArgs &a0, cudaStream_t s) {
    if (fn == c->k_batch_aff && fn != nullptr)
        return launch_geom(c, fn, ncand, a0, s, 256, 256, a0.H * (1 + c->dc.m) * c->dc.aff_np * 4, false);
    if (fn == c->k_batch)
        return launch_geom(c, fn, ncand, a0, s, c->bcand_per_block, c->bblock, c->bsmem, c->bpersistent);
    return launch_geom(c, fn, ncand, a0, s, c->cand_per_block, c->block, c->smem, c->variant == 2 || c->variant == 4);
}
cudaError_t launch_base(const mpmi_ctx *c, const KArgs &a, cudaStream_t s) {      // a_k = C K^k Psi(x_t) of the affine path
    void *args[2] = {(void *)&c->dc, (void *)&a};
    return cudaLaunchKernel((const void *)c->k_base, dim3((unsigned)c->dc.H), dim3(128), args, 0, s);
}

// one tick on stream s: [cell histogram + scan, scatter] (large Philox sets only) -> fused tick kernel
template <int NP>
const void *pick_predict_m(int m) {
    return m == 1 ? (const void *)bin_predict_kernel<NP, 1> : m == 2 ? (const void *)bin_predict_kernel<NP, 2>
         : m == 3 ? (const void *)bin_predict_kernel<NP, 3> : (const void *)bin_predict_kernel<NP, 4>;
}
const void *pick_predict(int np, int m) { return np == 4 ? pick_predict_m<4>(m) : np == 8 ? pick_predict_m<8>(m) : pick_predict_m<16>(m); }
unsigned pred_smem(const mpmi_ctx *c) { return (unsigned)(c->dc.H * (1 + c->dc.m) * c->dc.aff_np * 4 + (c->dc.H + 1) * 4); }   // table + CTA histogram
unsigned pred_grid(const mpmi_ctx *c) { return (unsigned)((c->bin.nsamp + 256 * kPredCand - 1) / (256 * kPredCand)); }
// scatter of the binning pass: cells from the Philox words, or (life-time order) from the predicted keys
const void *scatter_fn(const mpmi_ctx *c) { return c->predict ? (const void *)bin_scatter_keys_kernel : (const void *)bin_scatter_kernel; }
unsigned scatter_smem(const mpmi_ctx *c) { return c->predict ? (unsigned)(2 * c->bin.ncells * sizeof(int)) : 0u; }
unsigned scatter_grid(const mpmi_ctx *c, unsigned bin_grid) {
    if (!c->predict) return bin_grid;
    const long long g = (c->bin.nsamp + 1023) / 1024, gmax = 8LL * c->sm_count;
    return (unsigned)(g < gmax ? g : gmax);
}

#define CL(call) do { const cudaError_t e_ = (call); if (e_ != cudaSuccess) return e_; } while (0)
// bound kernels of the verified tensor-core tick (bound.cuh): E[j][r] for this x_t, then tau_i(k)
template <int D> const void *pick_btau(int np) {
    return np == 4 ? (const void *)bound_tau_kernel<D, 4> : np == 8 ? (const void *)bound_tau_kernel<D, 8> : (const void *)bound_tau_kernel<D, 16>;
}
cudaError_t launch_bound(const mpmi_ctx *c, const KArgs &a, cudaStream_t s) {
    void *eargs[2] = {(void *)&c->dc, (void *)&a};
    CL(cudaLaunchKernel(c->k_berr, dim3((unsigned)c->dc.H), dim3(c->berr_block), eargs, 0, s));
    void *targs[1] = {(void *)&c->dc};
    return cudaLaunchKernel(c->k_btau, dim3((unsigned)c->dc.H), dim3(kBoundTauThreads), targs, 0, s);
}
// second pass of the verified tick / batch: the FP32 kernel over the deferral lists
cudaError_t launch_recheck(const mpmi_ctx *c, KernFn fn, KArgs a, cudaStream_t s) {
    a.perm = nullptr; a.nsamp = 0; a.recheck_mode = 1 | (c->rc_warps << 8); a.kslot = c->kslot; a.st = c->d_state;
    a.work = c->recheck_persistent ? &c->d_state->work : nullptr;
    void *args[2] = {(void *)&c->dc, (void *)&a};
    return cudaLaunchKernel((const void *)fn, dim3(c->recheck_grid), dim3((unsigned)c->recheck_block), args, (size_t)c->recheck_smem, s);
}

cudaError_t enqueue_tick(const mpmi_ctx *c, KArgs a, cudaStream_t s) {
    // fork: the bound kernels need only x_t; they run on the context's side stream beside the binning kernels
    const bool fork = c->k_recheck && c->binning;
    if (c->k_recheck) {
        if (fork) {
            CL(cudaEventRecord(c->ev_fork, s));
            CL(cudaStreamWaitEvent(c->side, c->ev_fork, 0));
            CL(launch_bound(c, a, c->side));
            CL(cudaEventRecord(c->ev_join, c->side));
        } else {
            CL(launch_bound(c, a, s));
        }
    }
    if (c->binning) {
        BinArgs b = c->bin;
        b.tick_val = a.tick_val;
        long long g = (b.nsamp + 255) / 256;
        const long long gmax = 8LL * c->sm_count;
        const unsigned grid = (unsigned)(g < gmax ? g : gmax);
        void *pargs[2] = {(void *)&c->dc, (void *)&b};
        if (c->predict) {        // a_k for this x_t, then predicted life times (keys) + their histogram + scan
            CL(launch_base(c, a, s));
            CL(cudaLaunchKernel(c->k_pred, dim3(pred_grid(c)), dim3(256), pargs, pred_smem(c), s));
        } else {
            CL(cudaLaunchKernel((const void *)bin_hist_kernel, dim3(grid), dim3(256), pargs, 0, s));
        }
        CL(cudaLaunchKernel(scatter_fn(c), dim3(scatter_grid(c, grid)), dim3(256), pargs, scatter_smem(c), s));
        a.perm = c->d_perm; a.nsamp = b.nsamp;
    }
    if (c->affine) CL(launch_base(c, a, s));
    if (c->k_recheck) {
        a.recheck = c->d_recheck; a.recheck_count = c->d_recheck_count; a.recheck_mode = 0; a.recheck_tau_scale = c->recheck_tau_scale;
        if (fork) CL(cudaStreamWaitEvent(s, c->ev_join, 0));
    }
    a.timeline = c->timeline;
    cudaEvent_t *pe = c->prof ? const_cast<cudaEvent_t *>(&c->prof_ev[3 * (c->prof_n % kProfRing)]) : nullptr;
    if (pe) CL(cudaEventRecord(pe[0], s));
    CL(launch(c, c->k_tick, c->dc.shard_count, a, s));
    if (pe) CL(cudaEventRecord(pe[1], s));
    if (c->k_recheck) CL(launch_recheck(c, c->k_recheck, a, s));
    if (pe) { CL(cudaEventRecord(pe[2], s)); const_cast<mpmi_ctx *>(c)->prof_n++; }
    return cudaSuccess;
}
#undef CL

unsigned grid_for(const mpmi_ctx *c, long long ncand) {
    long long blocks = (ncand + c->cand_per_block - 1) / c->cand_per_block;
    if (blocks < 1) blocks = 1;
    if ((c->variant == 2 || c->variant == 4) && blocks > (long long)c->sm_count * c->tc_ctas) blocks = (long long)c->sm_count * c->tc_ctas;
    if (c->variant == 3 && c->lat_cap > 0 && blocks > c->lat_cap) blocks = c->lat_cap;
    return (unsigned)blocks;
}

void tick_node_params(mpmi_ctx *c, cudaKernelNodeParams *p, void **args) {
    std::memset(p, 0, sizeof *p);
    args[0] = (void *)&c->dc; args[1] = (void *)&c->ga;
    p->func = (void *)c->k_tick; p->gridDim = dim3(c->tick_grid); p->blockDim = dim3((unsigned)c->block);
    p->sharedMemBytes = (unsigned)c->smem; p->kernelParams = args;
}
void base_node_params(mpmi_ctx *c, cudaKernelNodeParams *p, void **args) {
    std::memset(p, 0, sizeof *p);
    args[0] = (void *)&c->dc; args[1] = (void *)&c->ga;
    p->func = (void *)c->k_base; p->gridDim = dim3((unsigned)c->dc.H); p->blockDim = dim3(128); p->kernelParams = args;
}
void pred_node_params(mpmi_ctx *c, cudaKernelNodeParams *p, void **args) {
    std::memset(p, 0, sizeof *p);
    args[0] = (void *)&c->dc; args[1] = (void *)&c->gb;
    p->func = (void *)c->k_pred; p->gridDim = dim3(pred_grid(c)); p->blockDim = dim3(256);
    p->sharedMemBytes = pred_smem(c); p->kernelParams = args;
}
void bin_node_params(mpmi_ctx *c, bool scatter, cudaKernelNodeParams *p, void **args) {
    std::memset(p, 0, sizeof *p);
    args[0] = (void *)&c->dc; args[1] = (void *)&c->gb;
    p->func = scatter ? (void *)scatter_fn(c) : (void *)bin_hist_kernel;
    p->gridDim = dim3(scatter ? scatter_grid(c, c->bin_grid) : c->bin_grid); p->blockDim = dim3(256); p->kernelParams = args;
    p->sharedMemBytes = scatter ? scatter_smem(c) : 0u;
}

void recheck_node_params(mpmi_ctx *c, cudaKernelNodeParams *p, void **args) {
    c->gr = c->ga;                               // same inputs, sequence number and result slot as the tick node
    c->gr.perm = nullptr; c->gr.nsamp = 0; c->gr.recheck_mode = 1 | (c->rc_warps << 8);
    c->gr.work = c->recheck_persistent ? &c->d_state->work : nullptr;
    std::memset(p, 0, sizeof *p);
    args[0] = (void *)&c->dc; args[1] = (void *)&c->gr;
    p->func = (void *)c->k_recheck; p->gridDim = dim3(c->recheck_grid); p->blockDim = dim3((unsigned)c->recheck_block);
    p->sharedMemBytes = (unsigned)c->recheck_smem; p->kernelParams = args;
}
void berr_node_params(mpmi_ctx *c, cudaKernelNodeParams *p, void **args) {
    std::memset(p, 0, sizeof *p);
    args[0] = (void *)&c->dc; args[1] = (void *)&c->ga;
    p->func = (void *)c->k_berr; p->gridDim = dim3((unsigned)c->dc.H); p->blockDim = dim3(c->berr_block); p->kernelParams = args;
}
void btau_node_params(mpmi_ctx *c, cudaKernelNodeParams *p, void **args) {
    std::memset(p, 0, sizeof *p);
    args[0] = (void *)&c->dc;
    p->func = (void *)c->k_btau; p->gridDim = dim3((unsigned)c->dc.H); p->blockDim = dim3(kBoundTauThreads); p->kernelParams = args;
}

int build_graph(mpmi_ctx *c) {
    c->ga = KArgs{};
    c->ga.st = c->d_state; c->ga.out = c->d_res_mapped; c->ga.inline_inputs = 1; c->ga.kslot = c->kslot;
    if (c->k_recheck) {
        c->ga.recheck = c->d_recheck; c->ga.recheck_count = c->d_recheck_count; c->ga.recheck_tau_scale = c->recheck_tau_scale;
        c->ga.deferred_out = c->d_deferred_mapped;
    }
    if (c->variant == 2 || c->variant == 4) c->ga.work = &c->d_state->work;
    c->tick_grid = grid_for(c, c->dc.shard_count);
    CU(c, cudaGraphCreate(&c->graph, 0));
    cudaKernelNodeParams p; void *args[2];
    cudaGraphNode_t dep = nullptr;
    if (c->binning) {
        c->gb = c->bin;
        long long g = (c->gb.nsamp + 255) / 256;
        const long long gmax = 8LL * c->sm_count;
        c->bin_grid = (unsigned)(g < gmax ? g : gmax);
        c->ga.perm = c->d_perm; c->ga.nsamp = c->gb.nsamp;
        if (c->predict) {                        // base -> prediction (keys + histogram + scan) -> scatter -> tick
            base_node_params(c, &p, args);
            CU(c, cudaGraphAddKernelNode(&c->n_base, c->graph, nullptr, 0, &p));
            pred_node_params(c, &p, args);
            CU(c, cudaGraphAddKernelNode(&c->n_hist, c->graph, &c->n_base, 1, &p));
        } else {
            bin_node_params(c, false, &p, args);
            CU(c, cudaGraphAddKernelNode(&c->n_hist, c->graph, nullptr, 0, &p));
        }
        bin_node_params(c, true, &p, args);
        CU(c, cudaGraphAddKernelNode(&c->n_scatter, c->graph, &c->n_hist, 1, &p));
        dep = c->n_scatter;
    }
    cudaGraphNode_t deps[3]; int ndep = 0;
    if (dep) deps[ndep++] = dep;
    if (c->k_recheck) {                          // bound kernels: a branch of their own beside the binning nodes
        berr_node_params(c, &p, args);
        CU(c, cudaGraphAddKernelNode(&c->n_berr, c->graph, nullptr, 0, &p));
        btau_node_params(c, &p, args);
        CU(c, cudaGraphAddKernelNode(&c->n_btau, c->graph, &c->n_berr, 1, &p));
        deps[ndep++] = c->n_btau;
    }
    if (c->affine) {                             // independent of the binning nodes: runs beside them
        base_node_params(c, &p, args);
        CU(c, cudaGraphAddKernelNode(&c->n_base, c->graph, nullptr, 0, &p));
        deps[ndep++] = c->n_base;
    }
    tick_node_params(c, &p, args);
    CU(c, cudaGraphAddKernelNode(&c->n_tick, c->graph, ndep ? deps : nullptr, ndep, &p));
    if (c->k_recheck) {
        recheck_node_params(c, &p, args);
        CU(c, cudaGraphAddKernelNode(&c->n_recheck, c->graph, &c->n_tick, 1, &p));
    }
    CU(c, cudaGraphInstantiate(&c->exec, c->graph, 0));
    return MPMI_OK;
}

}  // namespace

extern "C" {

const char *mpmi_strerror(int status) {
    switch (status) {
        case MPMI_OK: return "ok";
        case MPMI_ERR_INVALID: return "invalid argument";
        case MPMI_ERR_UNSUPPORTED: return "unsupported configuration or device";
        case MPMI_ERR_CUDA: return "CUDA runtime error";
        case MPMI_ERR_NOMEM: return "out of memory";
    }
    return "unknown status";
}

const char *mpmi_last_error(const mpmi_ctx *ctx) { return ctx ? ctx->err.c_str() : g_create_err.c_str(); }

void mpmi_destroy(mpmi_ctx *c) {
    if (!c) return;
    cudaSetDevice(c->device);
    if (c->pending) cudaStreamSynchronize(c->pending_stream);
    if (c->exec) cudaGraphExecDestroy(c->exec);
    if (c->graph) cudaGraphDestroy(c->graph);
    cudaFree(c->d_affM); cudaFree(c->d_KTa); cudaFree(c->d_W); cudaFree(c->d_b); cudaFree(c->d_terms);
    cudaFree(c->d_state);
    slot_release(c->device, c->kslot);
    cudaFree(c->d_affA); cudaFree(c->d_affG);
    cudaFree(c->d_pred);
    cudaFree(c->d_recheck); cudaFree(c->d_recheck_count);
    cudaFree(c->d_bnd_kpow); cudaFree(c->d_bnd_mid); cudaFree(c->d_bnd_econst); cudaFree(c->d_bnd_w); cudaFree(c->d_bnd_e); cudaFree(c->d_bnd_tau);
    if (c->ev_fork) cudaEventDestroy(c->ev_fork);
    if (c->ev_join) cudaEventDestroy(c->ev_join);
    if (c->side) cudaStreamDestroy(c->side);
    for (cudaEvent_t e : c->prof_ev) cudaEventDestroy(e);
    cudaFree(c->d_hist); cudaFree(c->d_cursor); cudaFree(c->d_perm); cudaFree(c->d_bin_ticket);
    cudaFreeHost(c->h_res);
    delete c;
}

int mpmi_create(const mpmi_config *cfg, mpmi_ctx **out) {
    g_create_err.clear();
    if (!cfg || !out) return fail(nullptr, MPMI_ERR_INVALID, "null config or output pointer");
    *out = nullptr;
    const int n = cfg->n, m = cfg->m, d = cfg->d;
    if (n <= 0 || m <= 0 || d <= 0 || cfg->N <= 0 || cfg->H <= 0) return fail(nullptr, MPMI_ERR_INVALID, "n, m, d, N, H must be positive");
    if (m > MPMI_MAX_M || n > MPMI_MAX_N || d > MPMI_MAX_D) return fail(nullptr, MPMI_ERR_UNSUPPORTED, "m > 4, n > 16 or d > 128");
    if (n > d) return fail(nullptr, MPMI_ERR_INVALID, "n > d: the first n lifted features must be the state");
    if (cfg->N > MPMI_MAX_CAND || cfg->H > 65535) return fail(nullptr, MPMI_ERR_UNSUPPORTED, "N or H too large");
    if (!cfg->K || !cfg->B || !cfg->u_lo || !cfg->u_hi) return fail(nullptr, MPMI_ERR_INVALID, "null K, B, u_lo or u_hi");
    if (!all_finite(cfg->K, (size_t)d * d) || !all_finite(cfg->B, (size_t)d * m)) return fail(nullptr, MPMI_ERR_INVALID, "non-finite K or B");
    if (!all_finite(cfg->u_lo, m) || !all_finite(cfg->u_hi, m)) return fail(nullptr, MPMI_ERR_INVALID, "non-finite input box");
    if (!std::isfinite(cfg->noise_sigma) || cfg->noise_sigma < 0.f) return fail(nullptr, MPMI_ERR_INVALID, "noise_sigma must be finite and >= 0");
    if (cfg->model != MPMI_MODEL_LINEAR && cfg->model != MPMI_MODEL_RELIFT) return fail(nullptr, MPMI_ERR_INVALID, "unknown model kind");
    for (int j = 0; j < m; j++) if (cfg->u_lo[j] > cfg->u_hi[j]) return fail(nullptr, MPMI_ERR_INVALID, "u_lo > u_hi");
    if (cfg->sampler != MPMI_SAMPLER_PHILOX && cfg->sampler != MPMI_SAMPLER_GRID) return fail(nullptr, MPMI_ERR_INVALID, "unknown sampler");
    if (cfg->sampler == MPMI_SAMPLER_GRID) {
        if (!cfg->grid_counts) return fail(nullptr, MPMI_ERR_INVALID, "grid sampler without grid_counts");
        long long prod = 1;
        for (int j = 0; j < m; j++) {
            if (cfg->grid_counts[j] <= 0) return fail(nullptr, MPMI_ERR_INVALID, "grid count <= 0");
            prod *= cfg->grid_counts[j];
            if (prod > MPMI_MAX_CAND) break;
        }
        if (prod != cfg->N) return fail(nullptr, MPMI_ERR_INVALID, "N != product of grid_counts");
    }
    const mpmi_lift_spec &L = cfg->lift;
    if (L.kind == MPMI_LIFT_MONO) {
        if (!L.terms) return fail(nullptr, MPMI_ERR_INVALID, "MONO lift without terms");
        for (int f = 0; f < d; f++)
            for (int q = 0; q < 4; q++) {
                const unsigned code = L.terms[4 * f + q];
                if (code != 0xFF && ((code >> 6) > 2 || (int)(code & 0x3F) >= n)) return fail(nullptr, MPMI_ERR_INVALID, "bad lift factor code");
            }
        for (int j = 0; j < n; j++)
            if (L.terms[4 * j] != j || L.terms[4 * j + 1] != 0xFF || L.terms[4 * j + 2] != 0xFF || L.terms[4 * j + 3] != 0xFF)
                return fail(nullptr, MPMI_ERR_INVALID, "the first n lift features must be the state itself");
    } else if (L.kind == MPMI_LIFT_RFF) {
        if (d > n && (!L.W || !L.b)) return fail(nullptr, MPMI_ERR_INVALID, "RFF lift without W or b");
        if (d > n && (!all_finite(L.W, (size_t)(d - n) * n) || !all_finite(L.b, d - n) || !std::isfinite(L.scale)))
            return fail(nullptr, MPMI_ERR_INVALID, "non-finite RFF table");
    } else {
        return fail(nullptr, MPMI_ERR_INVALID, "unknown lift kind");
    }
    const mpmi_safe_spec &S = cfg->safe;
    if (S.nbounds < 0 || S.nbounds > MPMI_MAX_BOUNDS || (S.nbounds > 0 && (!S.idx || !S.lo || !S.hi))) return fail(nullptr, MPMI_ERR_INVALID, "bad box constraints");
    for (int q = 0; q < S.nbounds; q++) {
        if (S.idx[q] < 0 || S.idx[q] >= n) return fail(nullptr, MPMI_ERR_INVALID, "box constraint index >= n");
        if (std::isnan(S.lo[q]) || std::isnan(S.hi[q])) return fail(nullptr, MPMI_ERR_INVALID, "NaN box limit");
    }
    if (!std::isfinite(S.inflate)) return fail(nullptr, MPMI_ERR_INVALID, "non-finite inflate");
    if (S.annulus) {
        if (S.ix < 0 || S.ix >= n || S.iy < 0 || S.iy >= n || S.ix == S.iy) return fail(nullptr, MPMI_ERR_INVALID, "bad annulus coordinates");
        if (!std::isfinite(S.cx) || !std::isfinite(S.cy) || !std::isfinite(S.rmin) || !std::isfinite(S.rmax) || S.rmin < 0)
            return fail(nullptr, MPMI_ERR_INVALID, "bad annulus radii");
    }
    const long long ncg = (long long)cfg->N + (cfg->include_user ? 1 : 0);
    long long sb = cfg->shard_begin, sc = cfg->shard_count;
    if (sb == 0 && sc == 0) sc = ncg;
    if (sb < 0 || sc <= 0 || sb + sc > ncg) return fail(nullptr, MPMI_ERR_INVALID, "shard outside [0, N + include_user]");

    int dev = cfg->device;
    if (dev < 0 && cudaGetDevice(&dev) != cudaSuccess) return fail(nullptr, MPMI_ERR_CUDA, "no CUDA device");
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, dev) != cudaSuccess) return fail(nullptr, MPMI_ERR_CUDA, "cudaGetDeviceProperties failed");
    if (prop.major != 10) return fail(nullptr, MPMI_ERR_UNSUPPORTED, "device is not compute capability 10.x (kernels are sm_100a only)");

    mpmi_ctx *c = new (std::nothrow) mpmi_ctx();
    if (!c) return fail(nullptr, MPMI_ERR_NOMEM, "host allocation failed");
    c->device = dev;
    if (const char *e = std::getenv("MPMI_RC_WARPS")) c->rc_warps = std::atoi(e) & 31;
    c->sm_count = prop.multiProcessorCount;
    int rc = MPMI_OK;
    auto bail = [&](int code) { g_create_err = c->err; mpmi_destroy(c); return code; };
    if (cudaSetDevice(dev) != cudaSuccess) { c->err = "cudaSetDevice failed"; return bail(MPMI_ERR_CUDA); }

    // ---- internal ordering of the physical dims: annulus coordinates, then box dims, then the rest
    DevCfg &dc = c->dc;
    std::memset(&dc, 0, sizeof dc);
    std::vector<int> perm;
    std::vector<char> used(n, 0);
    if (S.annulus) { perm.push_back(S.ix); perm.push_back(S.iy); used[S.ix] = used[S.iy] = 1; }
    for (int j = 0; j < n; j++) {
        bool boxed = false;
        for (int q = 0; q < S.nbounds; q++) boxed = boxed || S.idx[q] == j;
        if (boxed && !used[j]) { perm.push_back(j); used[j] = 1; }
    }
    for (int j = 0; j < n; j++) if (!used[j]) perm.push_back(j);
    auto po = [&](int f) { return f < n ? perm[f] : f; };

    const int D = d <= 8 ? 8 : d <= 16 ? 16 : d <= 32 ? 32 : d <= 64 ? 64 : 128;
    dc.n = n; dc.m = m; dc.d = d; dc.D = D;
    dc.N = cfg->N; dc.H = cfg->H; dc.include_user = cfg->include_user ? 1 : 0;
    dc.ncand_global = ncg; dc.shard_begin = sb; dc.shard_count = sc;
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

    // ---- augmented transposed model KTa[c][r]: c < D -> K[r][c], c >= D -> B[r][c-D]; zero padded
    const int M = m;
    std::vector<float> KTa((size_t)(D + M) * D, 0.f);
    for (int r = 0; r < d; r++) {
        for (int q = 0; q < d; q++) KTa[(size_t)q * D + r] = cfg->K[(size_t)po(r) * d + po(q)];
        for (int j = 0; j < m; j++) KTa[(size_t)(D + j) * D + r] = cfg->B[(size_t)po(r) * m + j];
    }
    std::vector<uint8_t> terms((size_t)D * 4, 0xFF);
    if (L.kind == MPMI_LIFT_MONO)
        for (int f = 0; f < d; f++) std::memcpy(&terms[4 * f], &L.terms[4 * po(f)], 4);

#define CUC(call) do { rc = [&]() -> int { CU(c, call); return MPMI_OK; }(); if (rc != MPMI_OK) return bail(rc); } while (0)
    CUC(cudaMalloc(&c->d_KTa, KTa.size() * sizeof(float)));
    CUC(cudaMemcpy(c->d_KTa, KTa.data(), KTa.size() * sizeof(float), cudaMemcpyHostToDevice));
    CUC(cudaMalloc(&c->d_terms, terms.size()));
    CUC(cudaMemcpy(c->d_terms, terms.data(), terms.size(), cudaMemcpyHostToDevice));
    if (L.kind == MPMI_LIFT_RFF && d > n) {
        CUC(cudaMalloc(&c->d_W, (size_t)(d - n) * n * sizeof(float)));
        CUC(cudaMemcpy(c->d_W, L.W, (size_t)(d - n) * n * sizeof(float), cudaMemcpyHostToDevice));
        CUC(cudaMalloc(&c->d_b, (size_t)(d - n) * sizeof(float)));
        CUC(cudaMemcpy(c->d_b, L.b, (size_t)(d - n) * sizeof(float), cudaMemcpyHostToDevice));
    }
    dc.KTa = c->d_KTa; dc.terms = c->d_terms; dc.W = c->d_W; dc.b = c->d_b;
    CUC(cudaMalloc(&c->d_state, sizeof(TickState)));
    TickState st0{kKeyNone, 0ull, 0u, 0u, 0u, 0u};
    CUC(cudaMemcpy(c->d_state, &st0, sizeof st0, cudaMemcpyHostToDevice));
    CUC(cudaHostAlloc(&c->h_res, sizeof(HostBlock), cudaHostAllocMapped));       // the result, then the second pass's count
    std::memset(c->h_res, 0, sizeof(HostBlock));
    CUC(cudaHostGetDevicePointer((void **)&c->d_res_mapped, c->h_res, 0));
    c->d_deferred_mapped = &reinterpret_cast<HostBlock *>(c->d_res_mapped)->deferred;

    // ---- kernel choice ------------------------------------------------------------------------------
    // prediction noise (Alg. 2 l.5) is built into the register, warp-tile, tensor-core (n <= 8) and re-lift kernels;
    // the latency kernel does not carry it, so sigma != 0 routes around it
    const bool noise = cfg->noise_sigma != 0.f;
    dc.noise_sigma = cfg->noise_sigma; dc.model = cfg->model;
    const int NPn = n <= 4 ? 4 : n <= 8 ? 8 : 16;
    const size_t aff_smem = (size_t)cfg->H * (1 + m) * NPn * sizeof(float);
    // tensor cores: linear lifted model only; noise block holds 8 dims; the verification tables (bound.cuh) must fit
    const bool tc_unverified = (cfg->variant & MPMI_VARIANT_TC_UNVERIFIED) != 0;
    const bool tc_model_ok = cfg->model == MPMI_MODEL_LINEAR && (!noise || n <= 8) &&
                             !(cfg->variant & (MPMI_VARIANT_NO_TENSOR | MPMI_VARIANT_AFFINE)) &&
                             (tc_unverified || ((size_t)cfg->H * D * D * sizeof(float) <= ((size_t)256 << 20) && aff_smem <= 200 * 1024));
    // ---- spatial binning: large Philox candidate sets only (the grid is already spatially ordered)
    {
        const long long send = sb + sc < cfg->N ? sb + sc : cfg->N;
        const long long nsamp = send > sb ? send - sb : 0;
        // measured at d = 32: the ~25 us of binning pay from 2^17 candidates for the register kernel (a warp of 64 candidates), from
        // ~80,000 for the tensor-core tick (a tile of 128 candidates runs until its last one stops)
        const bool tc32 = D == 32 && tc_model_ok && cfg->model == MPMI_MODEL_LINEAR;
        const bool want = cfg->sampler == MPMI_SAMPLER_PHILOX && nsamp >= (D > 32 ? (1 << 15) : tc32 ? kTc32MinBinning : (1 << 17));
        c->binning = (cfg->variant & MPMI_VARIANT_FORCE_BINNING) ? (cfg->sampler == MPMI_SAMPLER_PHILOX && nsamp >= 64)
                                                                  : (want && !(cfg->variant & MPMI_VARIANT_NO_BINNING));
        if (c->binning) {
            int total = 0;
            while ((64LL << (total + 1)) <= nsamp && total < 16) total++;      // ~64 candidates per cell
            for (int t = 0; t < total; t++) c->bin.bits[t % m]++;
            c->bin.ncells = 1 << total;
            c->bin.nsamp = nsamp;
            // (life-time order: H + 1 cells; padded to whole 64-cell groups for the scan's int4 accesses, the padding stays zero)
            const size_t ncell_alloc = (((size_t)(c->bin.ncells > cfg->H + 1 ? c->bin.ncells : cfg->H + 1) + 63) / 64) * 64;
            CUC(cudaMalloc(&c->d_hist, sizeof(int) * ncell_alloc));
            CUC(cudaMemset(c->d_hist, 0, sizeof(int) * ncell_alloc));
            CUC(cudaMalloc(&c->d_cursor, sizeof(int) * ncell_alloc));
            CUC(cudaMemset(c->d_cursor, 0, sizeof(int) * ncell_alloc));
            CUC(cudaMalloc(&c->d_perm, sizeof(int) * nsamp));
            CUC(cudaMalloc(&c->d_bin_ticket, sizeof(unsigned)));
            CUC(cudaMemset(c->d_bin_ticket, 0, sizeof(unsigned)));
            c->bin.hist = c->d_hist; c->bin.cursor = c->d_cursor; c->bin.perm = c->d_perm; c->bin.ticket = c->d_bin_ticket;
        }
    }

    bool tensor = false, tc32_batch = false;
    if (cfg->model == MPMI_MODEL_RELIFT) {
        // x' = C (K Psi(x) + B u): one thread per candidate, only the physical rows of the model (rollout_relift.cuh)
        c->variant = 5;
        c->P = 1; c->block = 128; c->cand_per_block = 128; c->smem = 0;
        c->bblock = c->block; c->bcand_per_block = c->cand_per_block;
        c->k_tick = mpmi_pick_relift(n, MODE_TICK);
        c->k_batch = mpmi_pick_relift(n, MODE_BATCH);
    } else if (D <= 32) {
        c->variant = 1;
        const int Pmax = 32 / D;
        // model source: the constant bank (one slot per context) when the grid fills the machine or the model fits the
        // immediate constant cache, shared memory otherwise (measured crossover at D = 32: ~2^19 candidates); the batch
        // kernels take the constant bank whenever a slot is free (it frees the LSU for the trajectory stores)
        c->kslot = (cfg->variant & MPMI_VARIANT_SMEM_MODEL) ? -1 : slot_acquire(dev);
        if (c->kslot >= 0 && set_model(D, noise, c->kslot, KTa.data(), (int)KTa.size()) != 0) {
            slot_release(dev, c->kslot); c->kslot = -1; (void)cudaGetLastError();
        }
        const int kconst_tick = (c->kslot >= 0 && ((D + M) * D * 4 <= 2048 || sc >= (1LL << 19))) ? 1 : 0;
        const int kconst_batch = c->kslot >= 0 ? 1 : 0;
        // shared-memory model: enough warps to give every SM sub-partition two warps at the wide packing?  else 2 cand/thread
        const long long warps_wide = (sc + 2LL * Pmax * 32 - 1) / (2LL * Pmax * 32);
        c->P = (cfg->variant & MPMI_VARIANT_NARROW) ? 1 : (cfg->variant & MPMI_VARIANT_WIDE) ? Pmax
               : kconst_tick ? 1 : (warps_wide >= 8LL * c->sm_count ? Pmax : 1);   // constant-bank model: 2 per thread is faster (measured)
        const long long threads = (sc + 2LL * c->P - 1) / (2LL * c->P);
        c->block = threads >= 128LL * 2 * c->sm_count ? 128 : threads >= 64LL * 2 * c->sm_count ? 64 : 32;
        c->cand_per_block = 2 * c->P * c->block;
        c->bblock = c->block; c->bcand_per_block = c->cand_per_block;
        c->smem = 0;
        c->k_tick = pick_reg(D, M, c->P, MODE_TICK, noise, kconst_tick);
        c->k_batch = pick_reg(D, M, c->P, MODE_BATCH, noise, kconst_batch);
        c->k_batch_dump = pick_reg(D, M, 1, MODE_BATCH, noise, kconst_batch);
        // paper-scale candidate sets: 4 lanes per candidate (rollout_lat.cuh) shorten the dependent chain
        const bool force_tc32 = D == 32 && tc_model_ok && (cfg->variant & MPMI_VARIANT_TENSOR32) &&
                                !(cfg->variant & (MPMI_VARIANT_NARROW | MPMI_VARIANT_WIDE | MPMI_VARIANT_LATENCY | MPMI_VARIANT_SMEM_MODEL));
        const bool lat = !noise && !force_tc32 && ((cfg->variant & MPMI_VARIANT_LATENCY) || (!(cfg->variant & (MPMI_VARIANT_NARROW | MPMI_VARIANT_WIDE)) && sc <= kLatMaxCand));
        if (lat && !c->binning) {
            // rows per lane: 2 (D/2 lanes per candidate) while that still leaves SMs short of warps, else 4
            const long long warps_r4 = sc * (D / 4) / 32;
            const int R = (cfg->variant & MPMI_VARIANT_LAT_R2) ? 2 : (cfg->variant & MPMI_VARIANT_LAT_R4) ? 4
                          : (warps_r4 < 4LL * c->sm_count ? 2 : 4);
            c->variant = 3;
            c->k_tick = pick_lat(D, M, R);
            c->block = 64; c->cand_per_block = 64 / (D / R);     // D/R lanes per candidate
            int occ = 0;
            if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, (const void *)c->k_tick, 64, 0) == cudaSuccess && occ > 0 && !std::getenv("MPMI_LAT_WAVES"))
                c->lat_cap = (long long)occ * c->sm_count;
        }
        // D = 32, large candidate sets: the 3xTF32 tcgen05 kernel of d = 128 with N = 32 MMAs and four CTAs per SM, as a
        // VERIFIED tick (below).  The batch entry stays on the FP32 register kernels chosen above.
        if (D == 32 && c->variant == 1 && tc_model_ok && (sc > kTc32CandPerCta * c->sm_count || (cfg->variant & MPMI_VARIANT_TENSOR32)) &&
            !(cfg->variant & (MPMI_VARIANT_NARROW | MPMI_VARIANT_WIDE | MPMI_VARIANT_LATENCY | MPMI_VARIANT_SMEM_MODEL))) {
            tensor = true;
            c->variant = 4;
            int threads = 0;
            c->k_tick = mpmi_pick_tc_tick(D, &c->smem, &threads, &c->tc_ctas, noise);
            c->block = threads; c->cand_per_block = 128;
            CUC(cudaFuncSetAttribute((const void *)c->k_tick, cudaFuncAttributeMaxDynamicSharedMemorySize, c->smem));
            if (tc_unverified) {         // measurement knob: the bare tensor-core kernel serves the batch entry as well
                int bs = 0, bt = 0, bc = 0;
                c->k_batch = mpmi_pick_tc_batch(D, &bs, &bt, &bc, noise);
                c->k_batch_dump = nullptr;
                c->bblock = bt; c->bcand_per_block = 128; tc32_batch = true;
                CUC(cudaFuncSetAttribute((const void *)c->k_batch, cudaFuncAttributeMaxDynamicSharedMemorySize, bs));
            }
        }
    } else {
        // d = 128: the step is a dense contraction -> 3xTF32 on the tcgen05 tensor cores (rollout_tc.cuh), verified (below),
        // unless the caller asks for the FP32 SIMT tile kernel; d = 64 stays on the SIMT tile kernel
        tensor = D == 128 && tc_model_ok;
        c->P = 1;
        int &fsmem = c->fp32_smem;
        c->k_batch_fp32 = pick_tile(D, M, MODE_BATCH, &fsmem, noise);
        if (tensor) {
            c->variant = 4;
            int threads = 0;
            c->k_tick = mpmi_pick_tc_tick(D, &c->smem, &threads, &c->tc_ctas, noise);
            c->k_batch = mpmi_pick_tc_batch(D, &c->smem, &threads, &c->tc_ctas, noise);
            c->block = threads; c->cand_per_block = 128;
        } else {
            c->variant = 2;
            c->block = kTileThreads; c->cand_per_block = kTileNC;
            c->k_tick = pick_tile(D, M, MODE_TICK, &c->smem, noise);
            c->k_batch = c->k_batch_fp32;
        }
        c->bblock = c->block; c->bcand_per_block = c->cand_per_block;
        if (c->k_tick) {
            CUC(cudaFuncSetAttribute((const void *)c->k_tick, cudaFuncAttributeMaxDynamicSharedMemorySize, c->smem));
            CUC(cudaFuncSetAttribute((const void *)c->k_batch, cudaFuncAttributeMaxDynamicSharedMemorySize, c->smem));
            CUC(cudaFuncSetAttribute((const void *)c->k_batch_fp32, cudaFuncAttributeMaxDynamicSharedMemorySize, fsmem));
        }
    }
    c->bsmem = (D <= 32 && !tc32_batch) ? 0 : c->smem;
    c->bpersistent = (c->variant == 2 || c->variant == 4) && (D > 32 || tc32_batch);
    // x_k = a_k + G_k u: tabulate G_k = C S_k B, S_k = sum_{i<k} K^i, in FP64 (T_1 = B, T_{k+1} = K T_k + B); a_k comes per tick
    // from affine_base_kernel.  Used by the affine variant and by the life-time order of the tile kernels.
    bool affine_built = false;
    auto build_affine = [&]() -> int {
        affine_built = true;
        const int Hh = cfg->H;
        std::vector<double> T((size_t)d * m), Tn((size_t)d * m);
        std::vector<float> G((size_t)Hh * m * NPn, 0.f);
        for (int r = 0; r < d; r++) for (int j = 0; j < m; j++) T[(size_t)r * m + j] = cfg->B[(size_t)r * m + j];
        for (int k = 0; k < Hh; k++) {
            for (int j = 0; j < m; j++)
                for (int q = 0; q < n; q++) G[((size_t)k * m + j) * NPn + q] = (float)T[(size_t)perm[q] * m + j];
            for (int r = 0; r < d; r++)
                for (int j = 0; j < m; j++) {
                    double sacc = cfg->B[(size_t)r * m + j];
                    for (int q = 0; q < d; q++) sacc += (double)cfg->K[(size_t)r * d + q] * T[(size_t)q * m + j];
                    Tn[(size_t)r * m + j] = sacc;
                }
            T.swap(Tn);
        }
        // rows of C K^k in the internal order of KTa: R_1 = first n rows of K, R_{k+1} = R_k K
        std::vector<float> Mt((size_t)Hh * NPn * D, 0.f);
        {
            std::vector<double> R((size_t)n * D, 0.0), Rn((size_t)n * D);
            for (int q = 0; q < n; q++) for (int cc = 0; cc < D; cc++) R[(size_t)q * D + cc] = KTa[(size_t)cc * D + q];
            for (int k = 0; k < Hh; k++) {
                for (int q = 0; q < n; q++) for (int cc = 0; cc < D; cc++) Mt[((size_t)k * NPn + q) * D + cc] = (float)R[(size_t)q * D + cc];
                if (k + 1 == Hh) break;
                std::fill(Rn.begin(), Rn.end(), 0.0);
                for (int q = 0; q < n; q++)
                    for (int r = 0; r < D; r++) {
                        const double v = R[(size_t)q * D + r];
                        if (v != 0.0) for (int cc = 0; cc < D; cc++) Rn[(size_t)q * D + cc] += v * (double)KTa[(size_t)cc * D + r];
                    }
                R.swap(Rn);
            }
        }
        CU(c, cudaMalloc(&c->d_affM, Mt.size() * sizeof(float)));
        CU(c, cudaMemcpy(c->d_affM, Mt.data(), Mt.size() * sizeof(float), cudaMemcpyHostToDevice));
        dc.aff_m = c->d_affM;
        CU(c, cudaMalloc(&c->d_affG, G.size() * sizeof(float)));
        CU(c, cudaMemcpy(c->d_affG, G.data(), G.size() * sizeof(float), cudaMemcpyHostToDevice));
        CU(c, cudaMalloc(&c->d_affA, (size_t)Hh * NPn * sizeof(float)));
        CU(c, cudaMemset(c->d_affA, 0, (size_t)Hh * NPn * sizeof(float)));
        dc.aff_g = c->d_affG; dc.aff_a = c->d_affA; dc.aff_np = NPn;
        c->k_base = mpmi_pick_affine_base(D);
        c->k_batch_aff = mpmi_pick_affine(NPn, MODE_BATCH);
        CU(c, cudaFuncSetAttribute((const void *)c->k_batch_aff, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)aff_smem));
        return MPMI_OK;
    };
    if ((cfg->variant & MPMI_VARIANT_AFFINE) && cfg->model == MPMI_MODEL_LINEAR && !noise && c->k_tick && c->k_batch &&
        aff_smem <= 200 * 1024) {
        rc = build_affine();
        if (rc != MPMI_OK) return bail(rc);
        c->affine = true; c->variant = 6;
        c->k_tick = mpmi_pick_affine(NPn, MODE_TICK);
        c->block = 256; c->cand_per_block = 256; c->smem = (int)aff_smem;
        CUC(cudaFuncSetAttribute((const void *)c->k_tick, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)aff_smem));
    } else if ((c->variant == 2 || c->variant == 4) && D > 32 && c->binning && cfg->model == MPMI_MODEL_LINEAR && !noise &&
               !(cfg->variant & MPMI_VARIANT_NO_PREDICT) && aff_smem <= 200 * 1024 && c->k_tick && c->k_batch) {
        // life-time order for the persistent tile kernels (binning.cuh): cells = predicted first-violation steps
        rc = build_affine();
        if (rc != MPMI_OK) return bail(rc);
        CUC(cudaMalloc(&c->d_pred, sizeof(int) * c->bin.nsamp));
        c->predict = true;
        c->k_pred = pick_predict(NPn, m);
        CUC(cudaFuncSetAttribute(c->k_pred, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)aff_smem + (cfg->H + 1) * 4));
        c->bin.keys = c->d_pred; c->bin.H = cfg->H; c->bin.ncells = cfg->H + 1;
    }
    // ---- verified tensor-core tick: second-pass kernel, deferral lists, bound tables (bound.cuh) -----------------------------
    if (tensor && c->variant == 4 && !tc_unverified) {
        if (!affine_built) { rc = build_affine(); if (rc != MPMI_OK) return bail(rc); }
        if (D == 32) {               // FP32 register kernel, 2 candidates per thread, CTAs loop over blocks of the lists
            const int rc_kconst = (c->kslot >= 0 && !std::getenv("MPMI_RC_SMEM")) ? 1 : 0;
            c->k_recheck = noise ? mpmi_pick_regn_32_recheck(M, rc_kconst) : mpmi_pick_reg_32_recheck(M, rc_kconst);
            // lanes per candidate pair in the second pass (measured, rollout_split.cuh): the fewer deferred candidates, the more the pass
            // is one warp's chain over the horizon -- 8 lanes up to ~300,000 candidates (40,000: tick 180 -> 164 us against 4 lanes, 2^16:
            // 192 -> 176, 2^17: 266 -> 255, 2^18: 376 -> 369, 2^19: 603 -> 620), 4 up to 2^19, 2 beyond
            // (0: one thread per pair, rollout_reg_kernel -- when the shared-memory model is forced, or MPMI_RC_RS=0)
            int rc_rs = sc <= 80000 ? 16 : sc <= 300000 ? 8 : sc <= (1LL << 19) ? 4 : 2;     // (16: 40,000 candidates 164 -> 157 us, 2^16 176 -> 173 us)
            if (const char *e = std::getenv("MPMI_RC_RS")) rc_rs = std::atoi(e);
            if (rc_rs == 2 || rc_rs == 4 || rc_rs == 8 || rc_rs == 16) {
                // row-split kernel, one-warp CTAs rolling blocks of 64 / RS candidates, 8 per SM: the pass is set by how long ONE
                // warp needs for the horizon, and RS lanes per pair cut that RS-fold (measured on C4, 3.8 % of 2^20 candidates:
                // one thread per pair 250 us however the blocks are dealt out)
                c->k_recheck = noise ? mpmi_pick_splitn_32(M, rc_rs) : mpmi_pick_split_32(M, rc_rs);
                c->recheck_block = 32; c->recheck_smem = 0; c->recheck_persistent = false;
                long long per_sm = 8;             // two persistent warps per sub-partition + first-come blocks (measured 4 / 6 / 8 / 10 / 16 per SM: 8 best at every N)
                if (const char *e = std::getenv("MPMI_RC_CTAS")) per_sm = std::atoi(e) > 0 ? std::atoi(e) : per_sm;   // (measurement aid)
                const long long per = 64 / rc_rs, nb = (sc + per - 1) / per, cap = per_sm * c->sm_count;
                c->recheck_grid = (unsigned)(nb < cap ? nb : cap);
            } else {
            // 4 one-warp CTAs per SM (one per sub-partition), each rolling blocks of 64 candidates: its own first, then first come,
            // first served (rollout_reg.cuh).
            c->recheck_block = 32; c->recheck_smem = 0; c->recheck_persistent = false;
            const long long nb = (sc + 63) / 64, cap = 4LL * c->sm_count;
            c->recheck_grid = (unsigned)(nb < cap ? nb : cap);
            }
        } else {                     // FP32 warp-tile kernel, persistent CTAs fetch batches of the lists from the work counter
            int bs = 0;
            c->k_recheck = noise ? mpmi_pick_tilen_128_tick_rc(M, &c->recheck_smem) : mpmi_pick_tile_128_tick_rc(M, &c->recheck_smem);
            c->k_batch_recheck = noise ? mpmi_pick_tilen_128_batch_rc(M, &bs) : mpmi_pick_tile_128_batch_rc(M, &bs);
            CUC(cudaFuncSetAttribute((const void *)c->k_batch_recheck, cudaFuncAttributeMaxDynamicSharedMemorySize, bs));
            c->recheck_block = kTileThreads; c->recheck_persistent = true;
            const long long nb = (sc + kTileNC / 2 - 1) / (kTileNC / 2);
            c->recheck_grid = (unsigned)(nb < c->sm_count ? nb : c->sm_count);
            CUC(cudaFuncSetAttribute((const void *)c->k_recheck, cudaFuncAttributeMaxDynamicSharedMemorySize, c->recheck_smem));
        }
        if (!c->k_recheck) { c->err = "no second-pass kernel for this (d, m)"; return bail(MPMI_ERR_UNSUPPORTED); }
        CUC(cudaMalloc(&c->d_recheck, sizeof(int) * (size_t)sc * kRecheckBuckets));
        CUC(cudaMalloc(&c->d_recheck_count, sizeof(unsigned) * (kRecheckBuckets + 1)));       // + the second pass's block counter
        CUC(cudaMemset(c->d_recheck_count, 0, sizeof(unsigned) * (kRecheckBuckets + 1)));
        if (const char *e = std::getenv("MPMI_TC_TAU_SCALE")) {
            const float v = (float)std::atof(e);
            if (v >= 0.f && v <= 16.f) c->recheck_tau_scale = v;
        }
        CUC(cudaStreamCreateWithFlags(&c->side, cudaStreamNonBlocking));
        CUC(cudaEventCreateWithFlags(&c->ev_fork, cudaEventDisableTiming));
        CUC(cudaEventCreateWithFlags(&c->ev_join, cudaEventDisableTiming));

        // -- tables, FP64, internal order (Kin[r][c] = KTa[c][r], Bin[r][j] = KTa[D + j][r])
        const int Hh = cfg->H;
        const double u24 = std::ldexp(1.0, -24);
        const int KB = D / 8;
        // column weights w_c of the per-step error bound E_r = sum_c w_c |K_rc| |z_c| (bound.cuh), internal column order:
        //   FP32 kernel: the FMA chain runs over the columns in DESCENDING order, so term c is rounded (c + 1) times, 2^-24 each
        //   (+1 when sigma*eps is added afterwards);
        //   3xTF32 operands: z_lo K_lo dropped (|z_lo| < 2^-10 |z|: the hardware truncates z_hi; |K_lo| <= 2^-11 |K|: K_hi is
        //   rounded to nearest): 2^-21; z_lo rounded to TF32 (2^-11 of a 2^-10 part): 2^-21; K_lo rounded (2^-11 of 2^-11): 2^-22;
        //   tensor-core accumulation: <= 2 ulp = 2^-22 of the running sum per MMA.  The full-magnitude Z_hi K_hi MMAs run input
        //   block, [noise block,] state blocks KB-1 .. 0: a product of state block b is followed by b + 1 accumulations, the
        //   input block by KB + 1 (+1 with noise); the 2 KB + 3 small-product MMAs before them run on sums below 2^-9 of the
        //   full magnitude: 2^-31 each.
        std::vector<float> wv((size_t)D + M, 0.f);
        const double w_operand = std::ldexp(1.0, -21) + std::ldexp(1.0, -21) + std::ldexp(1.0, -22);
        for (int cc = 0; cc < D + M; cc++) {
            const int nacc = cc < D ? cc / 8 + 1 : KB + 1 + (noise ? 1 : 0);
            wv[cc] = (float)(u24 * (cc + 1 + (noise ? 1 : 0)) + w_operand + std::ldexp(1.0, -22) * nacc + std::ldexp(1.0, -31) * (2 * KB + 3));
        }
        // the sigma*eps column: FP32 adds it with one rounding, the tensor-core path rounds sigma*eps itself, splits it (2^-21)
        // and accumulates it second of the full-magnitude MMAs
        const double wnoise = 2.0 * u24 + std::ldexp(1.0, -21) + std::ldexp(1.0, -22) * (KB + 1);
        const double epsmax = 5.77;                                                    // Box-Muller with u1 >= 2^-24: |eps| <= sqrt(48 ln 2) = 5.768
        std::vector<double> Kin((size_t)D * D), Bin((size_t)D * M);
        for (int r = 0; r < D; r++) {
            for (int cc = 0; cc < D; cc++) Kin[(size_t)r * D + cc] = KTa[(size_t)cc * D + r];
            for (int j = 0; j < M; j++) Bin[(size_t)r * M + j] = KTa[(size_t)(D + j) * D + r];
        }
        std::vector<double> umid(M), uhalf(M), umax(M);
        for (int j = 0; j < M; j++) {
            umid[j] = 0.5 * ((double)cfg->u_lo[j] + cfg->u_hi[j]); uhalf[j] = 0.5 * ((double)cfg->u_hi[j] - cfg->u_lo[j]);
            umax[j] = std::fmax(std::fabs((double)cfg->u_lo[j]), std::fabs((double)cfg->u_hi[j]));
        }
        std::vector<double> Kp((size_t)D * D, 0.0), Kn((size_t)D * D), T((size_t)D * M, 0.0), Tn((size_t)D * M), nz(D, 0.0), zabs(D);
        for (int r = 0; r < D; r++) Kp[(size_t)r * D + r] = 1.0;
        std::vector<float> kpowT((size_t)Hh * D * D), mid((size_t)Hh * D), econst((size_t)Hh * D);
        for (int j = 0; j < Hh; j++) {
            float *kt = &kpowT[(size_t)j * D * D];
            for (int r = 0; r < D; r++) for (int cc = 0; cc < D; cc++) kt[(size_t)cc * D + r] = (float)Kp[(size_t)r * D + cc];
            for (int r = 0; r < D; r++) {                       // z_j over the input box: centre (S_j B) u_mid, half-width |S_j B| u_half
                double mv = 0.0, av = 0.0;
                for (int i = 0; i < M; i++) { mv += T[(size_t)r * M + i] * umid[i]; av += std::fabs(T[(size_t)r * M + i]) * uhalf[i]; }
                mid[(size_t)j * D + r] = (float)mv;
                zabs[r] = av + (noise ? epsmax * (double)cfg->noise_sigma * nz[r] : 0.0);
            }
            for (int r = 0; r < D; r++) {
                double e = 0.0;
                for (int cc = 0; cc < D; cc++) e += (double)wv[cc] * std::fabs(Kin[(size_t)r * D + cc]) * zabs[cc];
                for (int i = 0; i < M; i++) e += (double)wv[D + i] * std::fabs(Bin[(size_t)r * M + i]) * umax[i];
                if (noise && r < n) e += wnoise * epsmax * (double)cfg->noise_sigma;
                econst[(size_t)j * D + r] = (float)(e * (1.0 + 1e-6));
            }
            if (j + 1 == Hh) break;
            if (noise) for (int r = 0; r < D; r++) for (int i = 0; i < n; i++) nz[r] += std::fabs(Kp[(size_t)r * D + i]);   // sum_{p<=j} |K^p E|
            std::fill(Kn.begin(), Kn.end(), 0.0);              // K^{j+1} = K K^j,  S_{j+1} B = K (S_j B) + B
            for (int r = 0; r < D; r++)
                for (int q = 0; q < D; q++) {
                    const double v = Kin[(size_t)r * D + q];
                    if (v != 0.0) for (int cc = 0; cc < D; cc++) Kn[(size_t)r * D + cc] += v * Kp[(size_t)q * D + cc];
                }
            Kp.swap(Kn);
            for (int r = 0; r < D; r++)
                for (int i = 0; i < M; i++) {
                    double v = Bin[(size_t)r * M + i];
                    for (int q = 0; q < D; q++) v += Kin[(size_t)r * D + q] * T[(size_t)q * M + i];
                    Tn[(size_t)r * M + i] = v;
                }
            T.swap(Tn);
        }
        auto up = [&](float **dst, const std::vector<float> &src) -> int {
            CU(c, cudaMalloc(dst, src.size() * sizeof(float)));
            CU(c, cudaMemcpy(*dst, src.data(), src.size() * sizeof(float), cudaMemcpyHostToDevice));
            return MPMI_OK;
        };
        if ((rc = up(&c->d_bnd_kpow, kpowT)) != MPMI_OK || (rc = up(&c->d_bnd_mid, mid)) != MPMI_OK ||
            (rc = up(&c->d_bnd_econst, econst)) != MPMI_OK || (rc = up(&c->d_bnd_w, wv)) != MPMI_OK) return bail(rc);
        CUC(cudaMalloc(&c->d_bnd_e, (size_t)Hh * D * sizeof(float)));
        CUC(cudaMalloc(&c->d_bnd_tau, (size_t)(Hh + 1) * (NPn + kTauPad) * sizeof(float)));
        CUC(cudaMemset(c->d_bnd_tau, 0, (size_t)(Hh + 1) * (NPn + kTauPad) * sizeof(float)));
        dc.bnd_kpow = c->d_bnd_kpow; dc.bnd_mid = c->d_bnd_mid; dc.bnd_econst = c->d_bnd_econst; dc.bnd_w = c->d_bnd_w;
        dc.bnd_e = c->d_bnd_e; dc.bnd_tau = c->d_bnd_tau;
        c->k_berr = D == 32 ? (const void *)bound_err_kernel<32> : (const void *)bound_err_kernel<128>;
        c->berr_block = D < 64 ? 64 : (unsigned)D;
        c->k_btau = D == 32 ? pick_btau<32>(NPn) : pick_btau<128>(NPn);
    }
    if (!c->k_tick || !c->k_batch) { c->err = "no kernel for this (d, m)"; return bail(MPMI_ERR_UNSUPPORTED); }
    cudaFuncAttributes fa;
    CUC(cudaFuncGetAttributes(&fa, (const void *)c->k_tick));
    c->regs = fa.numRegs;
    rc = build_graph(c);
    if (rc != MPMI_OK) return bail(rc);
#undef CUC
    *out = c;
    return MPMI_OK;
}

int mpmi_get_info(const mpmi_ctx *c, mpmi_info *o) {
    if (!c || !o) return MPMI_ERR_INVALID;
    std::memset(o, 0, sizeof *o);
    o->d_pad = c->dc.D; o->variant = c->variant; o->cand_per_block = c->cand_per_block;
    o->threads_per_block = c->block;
    o->blocks = (int)grid_for(c, c->dc.shard_count);
    o->smem_bytes = c->smem + (c->variant == 1 ? (c->dc.D + c->dc.m + 1) * c->dc.D * 4 : 0);
    o->regs_per_thread = c->regs; o->sm_count = c->sm_count; o->launches_per_tick = (c->binning ? 3 : 1) + (c->affine ? 1 : 0) + (c->predict ? 1 : 0) + (c->k_recheck ? 3 : 0); o->uses_graph = 1;
    o->binning_cells = c->binning ? c->bin.ncells : 0;
    o->ncand_local = c->dc.shard_count;
    if (c->k_recheck)                            // candidates the last finished HOST-path tick handed to the FP32 pass (mapped
        o->reserved = *reinterpret_cast<volatile const int *>(&reinterpret_cast<const HostBlock *>(c->h_res)->deferred);   // memory: no sync)
    return MPMI_OK;
}

int mpmi_step(mpmi_ctx *c, const float *x0, const float *u_user, uint64_t tick, void *stream) {
    if (!c) return MPMI_ERR_INVALID;
    if (!x0 || !u_user) return fail(c, MPMI_ERR_INVALID, "null x0 or u_user");
    if (!all_finite(x0, c->dc.n) || !all_finite(u_user, c->dc.m)) return fail(c, MPMI_ERR_INVALID, "non-finite x0 or u_user");
    CU(c, cudaSetDevice(c->device));
    if (c->pending) {                                       // one tick in flight per context
        mpmi_result drop;
        const int rc = mpmi_step_result(c, &drop);
        if (rc != MPMI_OK) return rc;
    }
    std::memcpy(c->ga.x0_val, x0, sizeof(float) * c->dc.n);
    std::memcpy(c->ga.u_val, u_user, sizeof(float) * c->dc.m);
    c->ga.tick_val = tick;
    if (++c->seq == 0) c->seq = 1;
    c->ga.seq = c->seq;
    // (a one-kernel tick goes through its one-node graph as well: measured on C1 / C2 / C3, cudaLaunchKernel with the ~1.2 KB of
    // by-value kernel parameters costs 10.3 us of host time per tick, node-parameter update + cudaGraphLaunch 6.5 us)
    cudaKernelNodeParams p; void *args[2];
    if (c->binning) {
        c->gb.tick_val = tick;
        if (c->predict) pred_node_params(c, &p, args); else bin_node_params(c, false, &p, args);
        CU(c, cudaGraphExecKernelNodeSetParams(c->exec, c->n_hist, &p));
        bin_node_params(c, true, &p, args);
        CU(c, cudaGraphExecKernelNodeSetParams(c->exec, c->n_scatter, &p));
    }
    if (c->affine || c->predict) {
        base_node_params(c, &p, args);
        CU(c, cudaGraphExecKernelNodeSetParams(c->exec, c->n_base, &p));
    }
    tick_node_params(c, &p, args);
    CU(c, cudaGraphExecKernelNodeSetParams(c->exec, c->n_tick, &p));
    if (c->k_recheck) {
        recheck_node_params(c, &p, args);
        CU(c, cudaGraphExecKernelNodeSetParams(c->exec, c->n_recheck, &p));
        berr_node_params(c, &p, args);
        CU(c, cudaGraphExecKernelNodeSetParams(c->exec, c->n_berr, &p));
    }
    CU(c, cudaGraphLaunch(c->exec, (cudaStream_t)stream));
    c->pending = true; c->pending_stream = (cudaStream_t)stream;
    c->err.clear();
    return MPMI_OK;
}

int mpmi_step_result(mpmi_ctx *c, mpmi_result *out) {
    if (!c || !out) return MPMI_ERR_INVALID;
    if (!c->pending) return fail(c, MPMI_ERR_INVALID, "no tick in flight");
    // the last CTA of the tick kernel writes the result into mapped pinned memory and then its sequence
    // number; poll for it (cheaper than a stream synchronise), checking the stream for errors now and then
    volatile mpmi_result *h = c->h_res;
    const int want = (int)c->seq;
    // back-off: a tight poll (with the CPU's spin-wait hint) for the first ~2^14 reads -- a paper-scale tick takes tens of
    // microseconds and the poll is what the latency harness times -- then the core is yielded between reads, and past ~2^20
    // reads (a tick that takes seconds: debugger, sanitizer, a time-sliced GPU) the thread sleeps 50 us per read
    for (unsigned spin = 0; h->reserved != want; spin++) {
        if ((spin & 0x3FFF) == 0x3FFF || spin >= (1u << 20)) {
            if (spin == 0xFFFFFFFFu) spin = 1u << 20;
            const cudaError_t e = cudaStreamQuery(c->pending_stream);
            if (e == cudaSuccess) { if (h->reserved != want) { c->pending = false; return fail(c, MPMI_ERR_CUDA, "tick finished without a result"); } break; }
            if (e != cudaErrorNotReady) { c->pending = false; c->err = std::string("tick failed: ") + cudaGetErrorString(e); return MPMI_ERR_CUDA; }
        }
        if (spin < (1u << 14)) cpu_relax();
        else if (spin < (1u << 20)) std::this_thread::yield();
        else std::this_thread::sleep_for(std::chrono::microseconds(50));
    }
    std::atomic_thread_fence(std::memory_order_acquire);
    c->pending = false;
    std::memcpy(out, c->h_res, sizeof *out);
    out->reserved = 0;
    return MPMI_OK;
}

int mpmi_step_sync(mpmi_ctx *c, const float *x0, const float *u_user, uint64_t tick, void *stream, mpmi_result *out) {
    if (!out) return MPMI_ERR_INVALID;
    const int rc = mpmi_step(c, x0, u_user, tick, stream);
    return rc != MPMI_OK ? rc : mpmi_step_result(c, out);
}

int mpmi_step_device(mpmi_ctx *c, const float *d_x0, const float *d_u_user, uint64_t tick, void *stream, mpmi_result *d_out) {
    if (!c) return MPMI_ERR_INVALID;
    if (!d_x0 || !d_u_user || !d_out) return fail(c, MPMI_ERR_INVALID, "null device pointer");
    CU(c, cudaSetDevice(c->device));
    KArgs a{};
    a.x0 = d_x0; a.u_user = d_u_user; a.tick_val = tick;
    a.st = c->d_state; a.out = d_out;
    CU(c, enqueue_tick(c, a, (cudaStream_t)stream));
    return MPMI_OK;
}

int mpmi_step_trace(mpmi_ctx *c, const float *d_x0, const float *d_u_user, uint64_t tick, void *stream, mpmi_result *d_out, int32_t *d_steps) {
    if (!c) return MPMI_ERR_INVALID;
    if (!d_x0 || !d_u_user || !d_out || !d_steps) return fail(c, MPMI_ERR_INVALID, "null device pointer");
    CU(c, cudaSetDevice(c->device));
    KArgs a{};
    a.x0 = d_x0; a.u_user = d_u_user; a.tick_val = tick;
    a.st = c->d_state; a.out = d_out; a.steps = d_steps;
    CU(c, enqueue_tick(c, a, (cudaStream_t)stream));
    return MPMI_OK;
}

int mpmi_profile_enable(mpmi_ctx *c, int32_t enable) {
    if (!c) return MPMI_ERR_INVALID;
    CU(c, cudaSetDevice(c->device));
    if (enable && c->prof_ev.empty()) {
        c->prof_ev.resize(3 * kProfRing, nullptr);
        for (cudaEvent_t &e : c->prof_ev) CU(c, cudaEventCreate(&e));
    }
    c->prof = enable != 0; c->prof_n = 0;
    return MPMI_OK;
}

int mpmi_profile_timeline(mpmi_ctx *c, uint64_t *d_stamps) {
    if (!c) return MPMI_ERR_INVALID;
    if (d_stamps && c->variant != 3) return fail(c, MPMI_ERR_UNSUPPORTED, "the stage timeline is recorded by the latency kernel (paper-scale candidate sets)");
    c->timeline = reinterpret_cast<unsigned long long *>(d_stamps);
    return MPMI_OK;
}

int mpmi_profile_read(mpmi_ctx *c, int32_t capacity, int32_t *count, float *ms_tick_kernel, float *ms_second_pass) {
    if (!c || !count || !ms_tick_kernel || !ms_second_pass || capacity <= 0) return MPMI_ERR_INVALID;
    CU(c, cudaSetDevice(c->device));
    const unsigned n = c->prof_n < kProfRing ? c->prof_n : kProfRing;
    int out = 0;
    for (unsigned i = c->prof_n - n; i < c->prof_n && out < capacity; i++, out++) {
        cudaEvent_t *pe = &c->prof_ev[3 * (i % kProfRing)];
        CU(c, cudaEventSynchronize(pe[2]));
        CU(c, cudaEventElapsedTime(&ms_tick_kernel[out], pe[0], pe[1]));
        CU(c, cudaEventElapsedTime(&ms_second_pass[out], pe[1], pe[2]));
    }
    *count = out;
    return MPMI_OK;
}

int mpmi_shard_step(mpmi_ctx *c, const float *d_x0, const float *d_u_user, uint64_t tick, void *stream, mpmi_partial *d_partial) {
    if (!c) return MPMI_ERR_INVALID;
    if (!d_x0 || !d_u_user || !d_partial) return fail(c, MPMI_ERR_INVALID, "null device pointer");
    CU(c, cudaSetDevice(c->device));
    KArgs a{};
    a.x0 = d_x0; a.u_user = d_u_user; a.tick_val = tick;
    a.st = c->d_state; a.out = nullptr; a.partial = d_partial;
    CU(c, enqueue_tick(c, a, (cudaStream_t)stream));
    return MPMI_OK;
}

int mpmi_shard_finalize(mpmi_ctx *c, const mpmi_partial *d_partials, int32_t G, const float *d_u_user, uint64_t tick,
                        void *stream, mpmi_result *d_out) {
    if (!c) return MPMI_ERR_INVALID;
    if (!d_partials || G <= 0 || !d_u_user || !d_out) return fail(c, MPMI_ERR_INVALID, "bad shard_finalize arguments");
    CU(c, cudaSetDevice(c->device));
    shard_finalise_kernel<<<1, 32, 0, (cudaStream_t)stream>>>(c->dc, d_partials, G, d_u_user, tick, d_out);
    CU(c, cudaGetLastError());
    return MPMI_OK;
}

int mpmi_rollout_batch(mpmi_ctx *c, const float *d_U, const float *d_X0, int64_t x0_count, int64_t Ncand, int32_t H,
                       int32_t dump_kind, float *d_traj, int32_t *d_steps, uint8_t *d_safe, uint64_t tick, void *stream) {
    if (!c) return MPMI_ERR_INVALID;
    if (!d_X0 || !d_steps) return fail(c, MPMI_ERR_INVALID, "null d_X0 or d_steps");
    if (Ncand <= 0 || Ncand > MPMI_MAX_CAND || H <= 0 || H > 65535) return fail(c, MPMI_ERR_INVALID, "bad Ncand or H");
    if (x0_count != 1 && x0_count != Ncand) return fail(c, MPMI_ERR_INVALID, "x0_count must be 1 or Ncand");
    if (dump_kind < MPMI_DUMP_NONE || dump_kind > MPMI_DUMP_LIFTED || (dump_kind != MPMI_DUMP_NONE && !d_traj))
        return fail(c, MPMI_ERR_INVALID, "bad dump_kind or null d_traj");
    CU(c, cudaSetDevice(c->device));
    KArgs a{};
    a.x0 = d_X0; a.u_user = nullptr; a.tick_val = tick;
    a.U = d_U; a.x0_count = x0_count; a.ncand = Ncand; a.H = H; a.dump_kind = dump_kind;
    a.traj = d_traj; a.steps = d_steps; a.safe = d_safe;
    if (c->affine && dump_kind != MPMI_DUMP_LIFTED && x0_count == 1 && H <= c->dc.H) {
        CU(c, launch_base(c, a, (cudaStream_t)stream));          // physical states only, shared x0: the affine path applies
        CU(c, launch(c, c->k_batch_aff, Ncand, a, (cudaStream_t)stream));
    } else if (dump_kind != MPMI_DUMP_NONE && c->k_batch_dump && c->variant != 5) {
        CU(c, launch_geom(c, c->k_batch_dump, Ncand, a, (cudaStream_t)stream, 256, 128, 0, false));
    } else if (c->k_batch_recheck) {
        // d = 128, verified context.  The bound tau_i(k) is taken over the context's input box, horizon and one x_t, so the
        // tensor-core batch applies to the internal sampler with a shared x0 (first pass: 3xTF32, every candidate; second
        // pass: the FP32 warp-tile kernel rewrites steps / flags / dumped states of the deferred ones); caller-supplied
        // inputs, per-candidate x0 or a longer horizon run on the FP32 warp-tile kernel alone.
        if (!d_U && x0_count == 1 && H <= c->dc.H && Ncand <= c->dc.shard_count) {
            cudaStream_t s = (cudaStream_t)stream;
            CU(c, launch_bound(c, a, s));
            a.recheck = c->d_recheck; a.recheck_count = c->d_recheck_count; a.recheck_mode = 0; a.recheck_tau_scale = c->recheck_tau_scale;
            CU(c, launch(c, c->k_batch, Ncand, a, s));
            CU(c, launch_recheck(c, c->k_batch_recheck, a, s));
        } else {
            CU(c, launch_geom(c, c->k_batch_fp32, Ncand, a, (cudaStream_t)stream, kTileNC, kTileThreads, c->fp32_smem, true));
        }
    } else {
        CU(c, launch(c, c->k_batch, Ncand, a, (cudaStream_t)stream));
    }
    return MPMI_OK;
}

}  // extern "C"

// kernel_args.cuh -- launch-time argument block shared by the host runtime and the kernels.
#pragma once
#include "mpmi_device.cuh"

namespace mpmi {

constexpr int kRegBlock = 128;
constexpr int kRecheckBuckets = 4;          // verified tensor-core tick: deferred candidates are listed per quarter of the horizon they survived

struct KArgs {
    // tick
    const float *x0;                      // device, n   (MODE_TICK; MODE_BATCH with x0_count == 1)
    const float *u_user;                  // device, m
    unsigned long long tick_val;
    // host path: the tick inputs travel BY VALUE inside the kernel-node parameters (no H2D copy node)
    float x0_val[kMaxN];
    float u_val[kMaxM];
    int inline_inputs;                    // 1: read x0_val / u_val instead of x0 / u_user
    int kslot;                            // constant-memory slot of this context's model (register kernels)
    unsigned seq;                         // written last into out->reserved (host polls it on mapped memory)
    TickState *st;
    mpmi_result *out;
    mpmi_partial *partial;
    const int *perm;                      // device, spatial order of the local sampled candidates, or null
    long long nsamp;                      // sampled candidates of this shard (perm entries)
    unsigned *work;                       // device batch counter of the persistent tile kernel (zero between launches)
    // verified tensor-core tick: candidates that came within tau_i(k) (bound.cuh) of the safe-set boundary in the 3xTF32
    // rollout are not keyed there but appended to `recheck`; the FP32 kernel (register kernel at D = 32, warp-tile kernel at
    // D = 128; recheck_mode = 1) rolls exactly those again, merges its keys into the same TickState and finalises the tick
    int *recheck;                         // device, kRecheckBuckets lists of capacity = local candidates each, or null
    unsigned *recheck_count;              // device, one per list; zeroed by the CTA that finalises
    int recheck_mode;                     // register kernel: 1 = walk the recheck lists (longest-lived first) instead of the index space
    float recheck_tau_scale;              // scales tau (1 = the derived bound; MPMI_TC_TAU_SCALE < 1 measures how conservative it is)
    int *deferred_out;                    // host-mapped: candidates the second pass rolled (mpmi_info.reserved), or null
    unsigned long long *timeline;         // device, 8 x gridDim %globaltimer stamps of the latency kernel's stages (mpmi_profile_timeline), or null
    // batch
    const float *U;                       // device Ncand*m or null
    long long x0_count;
    long long ncand;                      // candidates handled by this launch (local)
    int H;
    int dump_kind;
    float *traj;
    int *steps;
    uint8_t *safe;
};

// The augmented transposed model of the register kernels (D <= 32) lives in __constant__ memory, one slot per context
// (rollout_reg.cuh: c_model): K[r][c] then reaches FFMA2 as a uniform-register operand (LDCU on the uniform datapath)
// instead of through the LSU.  Measured: the same FFMA2 step loop runs at 96 % of the FP32 peak with the model in the
// constant bank against 88-90 % with warp-uniform LDS.128 (the LSU was the bound).  (A 4.6 KB by-value kernel parameter
// gives the same SASS but costs 160 s of cicc time per instantiation.)
constexpr int kModelSlots = 8;
constexpr int kModelFloats = (32 + kMaxM) * 32;

enum { MODE_TICK = 0, MODE_BATCH = 1 };

constexpr int kTileNC = 256;                      // candidates per CTA pass of the warp-tile kernel
constexpr int kTileThreads = 512;                 // = (kTileNC / 16 candidates per warp) * 32

}  // namespace mpmi

typedef void (*KernFn)(const mpmi::DevCfg, const mpmi::KArgs);

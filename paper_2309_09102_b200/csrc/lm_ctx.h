// lm_ctx.h -- private: the context behind the opaque lm_ctx of include/lm.h, shared by the
// translation units that implement the C ABI (lm_api.cu, lm_traj_api.cu).
#pragma once
#include "../../include/lm.h"
#include "lm_kernels.cuh"
#include "lm_traj.cuh"

#include <atomic>

namespace lmk {

struct Layout { // byte offsets into the workspace
    size_t q, lam, res, perr, rerr, its, mask, ui, us, conv, titers, totals, s_seeds, s_tp, s_tq, total;
};

struct TrajState { // trajectory-level LM (lm_traj_*), bound by lm_traj_attach
    bool attached = false;
    bool targets_packed = false;
    TArgs args{};
    float lambda0 = 1e-3f;
    int refine = 1;
    int cost_lanes = 0; // LM_OPT_TRAJ_COST_LANES: 0 = by shared_targets, 1 = lanes are trajectories, 2 = lanes are waypoints
    int fused_mode = 0; // LM_OPT_TRAJ_FUSED: 0 = by tile count, 1 = fused solve kernels, 2 = unfused (HBM) path
    size_t bytes = 0;
    char *ws = nullptr;
    size_t off_totals = 0, off_ui = 0, off_us = 0;
};

struct PlanState { // non-stationary schedule + anytime bookkeeping (lm_plan_*), bound by lm_plan_attach
    bool attached = false;
    lm_plan_params prm{};
    char *ws = nullptr;
    float *q_valid = nullptr;                 // [d][W] w-order
    float *cur = nullptr;                     // [6][B] max pos err, max rot err, mjac rev, mjac pris, length, min capsule clearance
    float *clear = nullptr;                   // [W] per-waypoint clearance (only with capsules)
    float *len_valid = nullptr;               // [B]
    int32_t *gate = nullptr, *first = nullptr, *records = nullptr; // [B]
    uint8_t *valid = nullptr;                 // [B]
    unsigned long long *total = nullptr;
};

int cuda_fail(cudaError_t e);              // records the error string for lm_strerror, returns LM_ECUDA
// lm_jit.cu: the LM kernel compiled at run time for one chain structure (lm_specialize)
int jit_get_kernel(const ChainSpec &s, bool fast, bool weighted, int var, bool hot, void **fn_out);
cudaError_t jit_launch(void *fn, unsigned grid, unsigned block, cudaStream_t s, const KArgs &a);
const char *jit_last_log();
std::atomic<long long> &launch_counter();  // lm_launch_count
inline size_t align_up(size_t x, size_t a = 256) { return (x + a - 1) / a * a; }
inline bool aligned16(const void *p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

} // namespace lmk

struct lm_ctx {
    int dof;
    int64_t B, n, W;
    int shared;
    lmk::KArgs args; // template for every launch
    lmk::Layout lay;
    char *ws;
    cudaStream_t stream;
    bool fresh;
    bool stale;       // lm_set_state injected q: res / pos_err / rot_err / frozen flag belong to the previous q until a launch
    int block;
    bool fast;
    int spec_id;      // structure-matched specialised kernel (lm_specs.cuh) or SPEC_GENERIC
    bool use_generic; // LM_OPT_GENERIC_KERNEL
    int lanes;        // LM_OPT_LANES_PER_WAYPOINT: 1 (default), 2 or 4
    lmk::ChainSpec sig; // structure of the chain (lm_api.cu: chain_signature)
    void *jit_fn;     // lm_specialize: the kernel compiled for `sig` (a CUfunction), nullptr = none
    bool jit_hot;     // ... as the HOT instantiation: only launched while refine == 1 and no trace is set
    lmk::TrajState traj;
    lmk::PlanState plan;
};

namespace lmk {
int materialize_state(lm_ctx *c);        // if nothing has run yet: state := seeds (a zero-iteration launch)
int refresh_waypoint_outputs(lm_ctx *c);
int reset_waypoint_lm_state(lm_ctx *c);  // lambda := lambda0, iters := 0, mask := 0 for every waypoint; q is kept
int launch_clearance(lm_ctx *c, float *clear_out); // lm_traj_api.cu
int run_pose_phase(lm_ctx *c, int max_iters); // = lm_run // zero-iteration launch: re-evaluates |r|, errors, frozen flag at the current q
}

#define LM_CUDA(x)                                        \
    do {                                                  \
        cudaError_t e_ = (x);                             \
        if (e_ != cudaSuccess) return lmk::cuda_fail(e_); \
    } while (0)

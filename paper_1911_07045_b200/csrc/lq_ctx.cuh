// lq_ctx.cuh -- the context behind the opaque lq_ctx handle and the small helpers every ABI source file uses
// (lq_api.cu: single-domain calls; lq_slab.cu: z-slab sub-domains).  Not part of the ABI.
#pragma once
#include "../../include/lq.h"
#include "lq_internal.cuh"
#include "lq_sweep.cuh"

#include <string>

struct lq_ctx {
    LqGeom g{};
    LqPhys ph{};
    int device = 0;
    cudaStream_t stream = nullptr;
    // state, padded SoA; [cur] is the live buffer, [cur^1] the sweep's output buffer
    double *q[2] = {nullptr, nullptr}, *v[2] = {nullptr, nullptr}, *F[2] = {nullptr, nullptr};
    int cur = 0;
    uint8_t *maskp = nullptr, *flags = nullptr, *kind = nullptr;
    double *W = nullptr, *axis = nullptr;
    bool flags_active = false, anch_active = false, has_Q = false;
    unsigned long long n_class[3] = {0, 0, 0};
    double *partials = nullptr;
    size_t partials_len = 0;
    double *dscal3 = nullptr;            // 3 doubles of energy output
    LqFireScalars *dsc = nullptr;        // 2 slots
    unsigned long long *dcounts = nullptr;
    int *dbad = nullptr;
    LqSweepPlan *sweep = nullptr;
    LqDescentPlan *descent = nullptr;
    // z-slab sub-domain (lq_create_slab): g.zopen = 1, the z ghost planes belong to the neighbour slabs
    int Lz_global = 0, z0 = 0;
    bool fire_open = false;              // between lq_fire_begin and lq_fire_end (step-wise FIRE of a sub-domain)
    LqFireConsts fire_fc{};
    long fire_sweeps = 0, fire_launches = 0;
    double *dtot = nullptr;              // 6 doubles: this sub-domain's reductions of the last lq_fire_step_local
    LqPartialSeg *dsegs = nullptr;       // device copy of the last sweep's partial-sum segments
    LqPartialSeg hsegs[3] = {};          // what dsegs holds (uploaded again only when a step's segments differ)
    int hnseg = -1;
    LqFireScalars **dscptr = nullptr;    // device array {&dsc[0]} for the advance kernel
    int fire_cur0 = 0, fire_buf = 0;     // live buffer when the run began / buffer the last sweep wrote
    bool fire_sweep_pending = false;     // lq_fire_step_local ran, lq_fire_step_finish not yet
    bool fire_last_first = false;        // the last sweep was the FIRST instantiation (its stop test is on q_0)
    int resident = 1;                    // "resident" option: small one-constant lattices run the on-chip kernel
    uint32_t *res_bond = nullptr;        // bond codes for the resident kernel (masked lattices)
    bool res_bond_dirty = true;
    int fire_path = 0;
    int rc_chunks = 0;                   // "rc_chunks" option: 0 = chunk table chosen by the makespan model
    bool v_valid = false;                // v[cur] holds the velocities of the last lq_fire_minimize (else: report zeros)
    double v_mix_a = 1.0, v_mix_b = 0.0; // FIRE rescale of the last step, not yet applied to v[cur] (the sweeps apply it lazily)
    cudaEvent_t ev0 = nullptr, ev1 = nullptr;   // timing of the minimisation loops (report.gpu_ms)
    void *scratch = nullptr;             // lq_analyze(LQ_HOST): device staging of the outputs, grown on demand
    size_t scratch_len = 0;
    std::string err;
};

extern thread_local std::string g_noctx_err;

inline int fail(lq_ctx *c, int code, const std::string &msg) {
    if (c) c->err = msg;
    else g_noctx_err = msg;
    return code;
}
#define LQ_CUDA(c, call)                                                                             \
    do {                                                                                             \
        cudaError_t e_ = (call);                                                                     \
        if (e_ != cudaSuccess)                                                                       \
            return fail((c), e_ == cudaErrorMemoryAllocation ? LQ_ERR_NOMEM : LQ_ERR_CUDA,           \
                        std::string(#call) + ": " + cudaGetErrorString(e_));                         \
    } while (0)

inline LqFields fields_of(const lq_ctx *c) {
    LqFields f;
    f.flags = c->flags_active ? c->flags : nullptr;
    f.kind = (c->flags_active && c->anch_active) ? c->kind : nullptr;
    f.W = c->W;
    f.axis = c->axis;
    return f;
}


// every ABI entry runs on the context's device, whatever device the calling thread had current
struct DeviceGuard {
    int prev = -1;
    explicit DeviceGuard(const lq_ctx *c) {
        if (c && cudaGetDevice(&prev) == cudaSuccess && prev != c->device) cudaSetDevice(c->device);
        else prev = -1;
    }
    ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};

inline bool bad_where(int w) { return w != LQ_HOST && w != LQ_DEVICE; }
int lq_ensure_field(lq_ctx *c, double **p);
// copy between a caller's dense [ncomp][nz][Ly][Lx] array (nz planes starting at padded z-plane index pz0) and a
// padded device array
cudaError_t lq_copy_box(const LqGeom &g, const void *padded, const void *user, size_t elem, int ncomp, bool to_padded,
                        cudaStream_t st, int pz0 = LQ_GH, int nz = -1, int user_z0 = 0, int user_nz = -1);

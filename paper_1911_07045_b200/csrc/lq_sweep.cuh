// lq_sweep.cuh -- interface of the fused force + FIRE sweep (lq_sweep.cu), the hot path.
#pragma once
#include "lq_internal.cuh"
#include <string>

struct LqSweepPlan;  // tensor maps, per-CTA partials, tile classification; owned by the context

void lq_sweep_destroy(LqSweepPlan *plan);
void lq_sweep_invalidate(LqSweepPlan *plan);  // geometry / anchoring arrays changed

// Runs up to max_steps FIRE steps, one kernel launch per step, INCLUDING Algorithm 1's initialisation (force of
// the initial state and the stop test on it): there is no separate first pass.  On entry buffer *cur holds q with
// its ghost shell valid (v and F need not be initialised) and dsc[0] the initial scalars (dt = dt0, alpha0,
// mix_a = mix_b = 0, step = 0; init = 1 for the stored path with velocity Verlet).  On return *cur is the buffer
// holding the final state, *h the final scalars.
// stored_F: true = state (q, vc, F), 240 B/site (any elastic constants); false = state (q, vc) with the force
// recomputed, 160 B/site (one-constant only; masked lattices included, no second kernel).
int lq_sweep_run(LqSweepPlan **plan, bool stored_F, const LqGeom &g, const LqPhys &ph, const LqFields &f, double *q[2],
                 double *v[2], double *F[2], int *cur, LqFireScalars *dsc, const LqFireConsts &fc, long max_steps,
                 cudaStream_t st, long *launches, long *sweeps, LqFireScalars *h, std::string &err, int rc_chunks = 0);

// The same in pieces (sub-domains, lq_slab.cu, drive several contexts step by step): build the plan; one sweep; the
// partial-sum segments that sweep left behind.
int lq_sweep_prepare(LqSweepPlan **plan, bool stored_F, const LqGeom &g, const LqPhys &ph, const LqFields &f, double *q[2],
                     double *v[2], double *F[2], cudaStream_t st, long *launches, std::string &err, int rc_chunks);
int lq_sweep_step(LqSweepPlan *plan, bool stored_F, const LqGeom &g, const LqPhys &ph, const LqFields &f, double *q[2],
                  double *v[2], double *F[2], int in, LqFireScalars *dsc, const LqFireConsts &fc, bool first, bool defer,
                  cudaStream_t st, std::string &err, int phase = 0);
int lq_sweep_segments(const LqSweepPlan *plan, bool stored_F, bool masked, bool first, LqPartialSeg seg[3]);

// gradient descent / Nesterov (lq_descent.cu): one launch per step; buf[0] holds q_0, nbuf rotating buffers
struct LqDescentPlan;
void lq_descent_destroy(LqDescentPlan *plan);
int lq_descent_run(LqDescentPlan **plan, int method, int path, const LqGeom &g, const LqPhys &ph, const LqFields &f,
                   double *const *buf, int nbuf, int *final, LqFireScalars *dsc, double eta, double mu,
                   double force_tol, long max_steps, cudaStream_t st, long *launches, long *sweeps,
                   LqFireScalars *h, std::string &err);

#include <cuda.h>
// 4-D tensor map (x, y, z, component) over a padded field with a bxw x byh x 1 x 5 box (lq_sweep.cu)
bool lq_make_box_map(CUtensorMap *m, const LqGeom &g, double *base, int bxw, int byh);
void lq_descent_invalidate(LqDescentPlan *plan);   // geometry / anchoring arrays changed

// recompute-F kernel (lq_sweep_rc.cu)
namespace lqsw { struct SweepArgs; }
int lq_sweep_rc_box(int which, int dim);
int lq_sweep_rc_tile(int dim);
int lq_sweep_rc_max_chunk();
// first: the first sweep of a call (velocity Verlet): also reduces the stop test on the initial state.
// attr_set[4]: per-plan record of which instantiations had their shared-memory attribute set (per device).
cudaError_t lq_launch_sweep_rc(bool masked, bool first, int ncta, bool *attr_set, const CUtensorMap &mq,
                               const CUtensorMap &mv, const lqsw::SweepArgs &a, cudaStream_t st);

// fix-up kernel for the non-plain sites of masked lattices (lq_fixup.cu)
int lq_fixup_build_list(const LqGeom &g, const uint8_t *flags, const uint8_t *plain, int **list, int *n, cudaStream_t st);
int lq_fixup_num_blocks(int n);
cudaError_t lq_launch_fixup(bool three, const LqGeom &g, const LqPhys &ph, const LqFields &f, const double *q,
                            double *v, double *F, const int *list, int n, LqFireScalars *sc, const LqFireConsts &fc,
                            const double *sweep_partials, int n_sweep, double *partials, unsigned int *counter,
                            cudaStream_t st, int defer = 0);

// FIRE with the state resident on chip: one cooperative launch per lq_fire_minimize call (lq_resident.cu)
bool lq_resident_plan(const LqGeom &g, int nsm, int dims[6]);
// q, v, F: ping-pong state buffers; step s reads buffer (cur + s) & 1 and writes the other, so the final state sits
// in buffer (cur + steps taken) & 1.  partials: 10 doubles per CTA.
cudaError_t lq_launch_fire_resident(const LqGeom &g, const LqPhys &ph, const LqFields &f, double *const q[2],
                                    double *const v[2], double *const F[2], int cur, const uint32_t *bond,
                                    LqFireScalars *sc, const LqFireConsts &fc, double *partials, const int dims[6],
                                    cudaStream_t st);

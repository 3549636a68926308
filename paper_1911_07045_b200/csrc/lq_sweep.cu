// lq_sweep.cu -- placeholder until the fused sweep lands
#include "lq_sweep.cuh"
#include "../../include/lq.h"
struct LqSweepPlan { int dummy; };
void lq_sweep_destroy(LqSweepPlan *p) { delete p; }
void lq_sweep_invalidate(LqSweepPlan *) {}
int lq_sweep_run(LqSweepPlan **, const LqGeom &, const LqPhys &, const LqFields &, double *[2], double *[2],
                 double *[2], int *, LqFireScalars *, const LqFireConsts &, long, cudaStream_t, long *, long *,
                 LqFireScalars *, std::string &err) {
    err = "fused sweep not built";
    return LQ_ERR_STATE;
}

// lq_internal.cuh -- shared declarations of the CUDA library (not part of the ABI).
//
// HBM layout.  Every per-site array lives in a PADDED box with a
// ghost shell of width LQ_GH that mirrors the periodic images, so no kernel does modular
// index arithmetic and TMA boxes with halos never wrap:
//     p(x,y,z) = (x + LQ_XO) + Px * ((y + LQ_GH) + Py * (z + LQ_GH))
// Px = roundup(LQ_XO + Lx + LQ_GH, 16): row starts and the first interior element of each
// row are 128-byte aligned; the low-x ghosts sit in the LQ_GH elements before it.
// Fields are SoA: component c of a 5-component field starts at c * NP.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

constexpr int LQ_GH = 2;   // ghost width in x, y and z
constexpr int LQ_XO = 16;  // element offset of x = 0 inside a padded row (128 B for fp64)

// Bond code of a site (one-constant masked sweeps; built once per lq_set_sites by k_bond_map): for the six directions
// d = (+x, -x, +y, -y, +z, -z) two bits at 2d index the weight a^s_k(x) [w_k(x) + w_k(x + s k)] of that bond in the
// gather-form force: 0 -> 0 (neighbour not simulated), 1 -> 1, 2 -> 3/2, 3 -> 2.
constexpr unsigned LQ_BOND_PLAIN = 0x555u;       // all six bonds at weight 1: the constant 7-point stencil
constexpr unsigned LQ_BOND_OBJECT = 1u << 12;    // the site itself is an object (no variables)
constexpr unsigned LQ_BOND_ANCH = 1u << 13;      // class boundary and kind != 0: an anchoring term applies
__host__ __device__ inline double lq_bond_weight(unsigned code, int d) {
    const unsigned i = (code >> (2 * d)) & 3u;
    return i == 0u ? 0.0 : 0.5 + 0.5 * (double)i;
}

struct LqGeom {
    int Lx, Ly, Lz;
    int Px, Py, Pz;
    long long sy, sz;  // strides (elements) of +y and +z in the padded box
    long long NP;      // padded sites per component
    long long N;       // Lx*Ly*Lz
    int gwx;           // width of the x ghost images the sweeps write: LQ_GH, or 4 where Lx % 4 == 0 and the row padding
                       // has room -- the images of x = 0..3 / Lx-4..Lx-1 then fill whole 32-byte sectors (a 16-byte
                       // store into a sector costs the ECC'd HBM a read-modify-write); cells beyond LQ_GH are never read
    int zopen;         // 1: z-slab sub-domain: the z ghost planes hold the neighbour slabs' planes
                       // (halo exchange), nothing wraps in z and no kernel writes z ghost images
    __host__ __device__ inline long long pidx(int x, int y, int z) const {
        return (long long)(x + LQ_XO) + sy * (long long)(y + LQ_GH) + sz * (long long)(z + LQ_GH);
    }
};

struct LqPhys {
    double A, B, C, L1, L2, L3, S0;
    // external fields, Eq. 13: T_ab = (chi H_a H_b + eps E_a E_b) / 3 in (xx,xy,xz,yy,yz,zz) order,
    // f_external = -T_ab Q_ab; Fx = the constant force it adds in the five stored variables (all 0 without a field)
    double T[6], Fx[5];
    double L4;   // chiral distortion constant of Eq. 10; 0 = off
    double L6;   // cubic distortion constant of Eq. 10; 0 = off
};
// the 19-point / general mixed-derivative code paths are needed as soon as any of L2, L3, L4 is non-zero
__host__ __device__ inline bool lq_three(const LqPhys &ph) { return ph.L2 != 0.0 || ph.L3 != 0.0 || ph.L4 != 0.0 || ph.L6 != 0.0; }

// FIRE state that lives on the device (Algorithm 1).
// mix_a, mix_b: the velocity rescale of the step just reduced, v <- mix_a*v + mix_b*F
// (mix_a = 1-alpha, mix_b = alpha*|v|/|F|; both 0 after a P <= 0 reset), applied lazily
// by the next sweep.  dt is the step size of the NEXT step.
struct LqFireScalars {
    double dt, alpha;
    double mix_a, mix_b;
    double P, FF, vv, Fmax;
    long long step;  // steps completed
    int npos;
    int converged;
    double dt_prev;  // semi-implicit Euler variant: the dt of the step just scheduled (its drift uses it)
    int init;        // 1: the next sweep is the initial force evaluation of the stored-force path (all step
                     // coefficients 0: q' = q, vc' = 0, F' = force(q)); its reduction only runs the stop test
};

struct LqFireConsts {
    double dt0, dtmax, alpha0, finc, fdec, falpha, force_tol;
    int Nmin;
    long long max_steps;
    int euler;  // 1: FIRE on the semi-implicit Euler step (integrator = 1), 0: velocity Verlet
};

// Reductions of one step -> schedule of the next (Algorithm 1; readings
// DESIGN.md R3, R12, R13).  tot = (P, |F|^2, |v|^2, max|F_a|).  first != 0: the initial force
// evaluation (ran with dt = 0, no kick): only the convergence test applies.
__host__ __device__ inline void lq_fire_advance(LqFireScalars &t, const LqFireConsts &fc, const double tot[4], int first) {
    t.P = tot[0]; t.FF = tot[1]; t.vv = tot[2]; t.Fmax = tot[3];
    if (first) t.dt = fc.dt0;
    else t.step += 1;
    if (t.Fmax < fc.force_tol) {
        t.converged = 1;
    } else if (!first) {
        if (t.FF > 0.0) { t.mix_a = 1.0 - t.alpha; t.mix_b = t.alpha * sqrt(t.vv / t.FF); }
        else { t.mix_a = 1.0; t.mix_b = 0.0; }
        if (t.P > 0.0) {
            t.npos += 1;
            if (t.npos > fc.Nmin) { t.dt = fmin(t.dt * fc.finc, fc.dtmax); t.alpha *= fc.falpha; }
        } else {
            t.npos = 0; t.dt *= fc.fdec; t.alpha = fc.alpha0; t.mix_a = 0.0; t.mix_b = 0.0;
        }
    }
}

// Same for FIRE on the semi-implicit Euler step (integrator = 1, R30).  tot are the reductions
// of (F(q_k), v after the full kick v += dt F).  The stop test reads F(q_k); a step is scheduled only while the
// budget lasts; the drift kernel then applies v <- mix_a v + mix_b F, q += dt_prev v.
__host__ __device__ inline void lq_fire_advance_euler(LqFireScalars &t, const LqFireConsts &fc, const double tot[4]) {
    t.FF = tot[1]; t.Fmax = tot[3];
    if (t.Fmax < fc.force_tol) { t.converged = 1; return; }
    if (t.step >= fc.max_steps) { t.mix_a = 1.0; t.mix_b = 0.0; t.dt_prev = 0.0; return; }
    t.step += 1;
    t.P = tot[0]; t.vv = tot[2];
    if (t.FF > 0.0) { t.mix_a = 1.0 - t.alpha; t.mix_b = t.alpha * sqrt(t.vv / t.FF); }
    else { t.mix_a = 1.0; t.mix_b = 0.0; }
    t.dt_prev = t.dt;
    if (t.P > 0.0) {
        t.npos += 1;
        if (t.npos > fc.Nmin) { t.dt = fmin(t.dt * fc.finc, fc.dtmax); t.alpha *= fc.falpha; }
    } else {
        t.npos = 0; t.dt *= fc.fdec; t.alpha = fc.alpha0; t.mix_a = 0.0; t.mix_b = 0.0;
    }
}

// The three coefficients a fused step needs, for either integrator (the lazily applied part of the previous step
// plus this step's kick):  v_k = ma vc + cF F ;  q' = q + dt v_k ;  vc' = v_k + kick F'.
//   velocity Verlet: dt = sc.dt, cF = mix_b + dt/2, kick = dt/2
//   Euler variant:   dt = sc.dt_prev (the scheduled step's own dt), cF = mix_b, kick = sc.dt while the budget lasts
struct LqStepCoef { double dt, ma, cF, kick; };
__host__ __device__ inline LqStepCoef lq_step_coef(const LqFireScalars &sc, const LqFireConsts &fc) {
    LqStepCoef k;
    if (sc.init) { k.dt = k.ma = k.cF = k.kick = 0.0; return k; }
    k.ma = sc.mix_a;
    if (fc.euler) { k.dt = sc.dt_prev; k.cF = sc.mix_b; k.kick = sc.step < fc.max_steps ? sc.dt : 0.0; }
    else { k.dt = sc.dt; k.cF = sc.mix_b + 0.5 * sc.dt; k.kick = 0.5 * sc.dt; }
    return k;
}
__host__ __device__ inline void lq_fire_advance_any(LqFireScalars &t, const LqFireConsts &fc, const double tot[4]) {
    if (fc.euler) lq_fire_advance_euler(t, fc, tot);
    else if (t.init) { lq_fire_advance(t, fc, tot, 1); t.init = 0; t.mix_a = 0.0; t.mix_b = 0.0; }
    else lq_fire_advance(t, fc, tot, 0);
}
// First sweep of the recompute path (velocity Verlet): its phase 1 evaluates F(q) of the INITIAL state anyway, so the
// stop test of Algorithm 1's initialisation ("if max|F| < tol return, steps = 0") rides on it:
// tot0 = (|F(q_0)|^2, max|F_a(q_0)|).  If it passes (or no step was asked for) the step this sweep computed is
// discarded (the caller does not flip buffers while step == 0); otherwise the step counts.
__host__ __device__ inline void lq_fire_advance_first(LqFireScalars &t, const LqFireConsts &fc, const double tot[4],
                                                      const double tot0[2]) {
    if (tot0[1] < fc.force_tol || fc.max_steps == 0) {
        t.P = 0.0; t.FF = tot0[0]; t.vv = 0.0; t.Fmax = tot0[1];
        t.converged = tot0[1] < fc.force_tol ? 1 : 0;
        return;
    }
    lq_fire_advance(t, fc, tot, 0);
}

struct LqFields {
    // padded device arrays; any of flags/kind/W/axis may be null (no objects / no anchoring)
    const uint8_t *flags;
    const uint8_t *kind;
    const double *W;
    const double *axis;  // [3][NP]
};

// ---- generic kernels (lq_kernels.cu) ----------------------------------------------------
double lq_measure_fp64_fma(int device, cudaStream_t st);   // fp64 FMA microbenchmark, TFLOP/s (< 0: error)
void lq_launch_fill_ghosts_f64(const LqGeom &g, double *field, int ncomp, cudaStream_t st);
void lq_launch_fill_ghosts_u8(const LqGeom &g, uint8_t *field, cudaStream_t st);
void lq_launch_classify(const LqGeom &g, const uint8_t *mask_p, uint8_t *flags_p, cudaStream_t st);
// sub-domains: mask_ext is a DENSE [Lz+6][Ly][Lx] array covering planes -3 .. Lz+2; flags are written on planes -2 .. Lz+1
void lq_launch_classify_ext(const LqGeom &g, const uint8_t *mask_ext, uint8_t *flags_p, cudaStream_t st);
// reductions of a step across sub-domains: seg[i] = (partials pointer, count, stride 4 | 2) in a fixed order
struct LqPartialSeg { const double *p; int n; int width; };
void lq_launch_reduce_partials(const LqPartialSeg *seg_dev, int nseg, double *tot6, cudaStream_t st);
// tot = nrank x 6 doubles (P, FF, vv, Fmax, FF0, Fmax0), combined in rank order; advances every sc[i] identically
void lq_launch_advance(const double *tot, int nrank, LqFireScalars *const *sc_dev, int nsc, LqFireConsts fc, int first,
                       cudaStream_t st);
void lq_launch_count_classes(const LqGeom &g, const uint8_t *flags_p, unsigned long long *counts3, cudaStream_t st);
void lq_launch_check_u8_max(const LqGeom &g, const uint8_t *arr_p, int maxval, int *bad, cudaStream_t st);
void lq_launch_check_dense_u8_max(const uint8_t *a, long long n, int maxval, int *bad, cudaStream_t st);
void lq_launch_check_dense_u8_ne(const uint8_t *a, long long n, int value, int *bad, cudaStream_t st);
void lq_launch_forces(const LqGeom &g, const LqPhys &ph, const LqFields &f, const double *q, double *F, cudaStream_t st);
// energy: partial sums per block into partials (3 per block) then final reduce into out3 (device)
int lq_energy_num_blocks(const LqGeom &g);
void lq_launch_energy(const LqGeom &g, const LqPhys &ph, const LqFields &f, const double *q,
                      double *partials, double *out3, cudaStream_t st);

// unfused FIRE path (fire_path = 1): 4 launches per step
int lq_fire1_num_blocks(const LqGeom &g);
// euler != 0 / euler_max >= 0: the semi-implicit Euler variant (full kick while sc->step < euler_max; drift with
// dt_prev and no half kick; first == 2 in lq_launch_fire_update)
void lq_launch_fire1_drift(const LqGeom &g, const LqFields &f, double *q, double *v, const double *F,
                           const LqFireScalars *sc, cudaStream_t st, int euler = 0);
void lq_launch_fire1_force(const LqGeom &g, const LqPhys &ph, const LqFields &f, const double *q, double *v,
                           double *F, const LqFireScalars *sc, double *partials, cudaStream_t st,
                           long long euler_max = -1);
void lq_launch_fire_update(const double *partials, int nblocks, LqFireScalars *sc_in_out, LqFireConsts fc,
                           int first, cudaStream_t st);
void lq_launch_zero_object_sites(const LqGeom &g, const uint8_t *flags, double *field, cudaStream_t st);
void lq_launch_analyze(const LqGeom &g, const double *q, const uint8_t *flags, double thr, double *S, double *dir,
                       uint8_t *defect, unsigned long long *count, cudaStream_t st);
void lq_launch_plain_map(const LqGeom &g, const uint8_t *flags, uint8_t *plain, cudaStream_t st);
void lq_launch_tile_summary(const LqGeom &g, const uint8_t *plain, uint8_t *tsum, int TX, int TY, int ntx, int nty,
                            cudaStream_t st);
void lq_launch_axpby(long long n, double a, const double *v, double b, const double *F, double *out, cudaStream_t st);
void lq_launch_bond_map(const LqGeom &g, const uint8_t *flags, const uint8_t *kind, uint32_t *bond, cudaStream_t st);
void lq_launch_tile_summary_bond(const LqGeom &g, const uint32_t *bond, uint8_t *tsum, int TX, int TY, int ntx, int nty,
                                 cudaStream_t st);

// lq_analyze.cu -- per-site analysis of a Q field: the headless counterpart of what the paper's
// GUI draws.  "The nematic director can be recovered as the eigenvector corresponding to the largest eigenvalue of
// Q, which equals S" (Eq. 2); defects are "regions where the largest eigenvalue of Q falls below some
// threshold".  One thread per site, streaming: reads 40 B (+1 flag byte), writes S (8 B),
// the director (24 B) and the defect byte; HBM-bound.
//
// Largest eigenvalue of the symmetric traceless 3x3 tensor in closed form (trigonometric solution of the
// depressed cubic lambda^3 - (p2/2) lambda - det = 0, p2 = tr Q^2; seeded in fp32), polished to fp64 by Newton steps
// on the characteristic polynomial; eigenvector = the largest cross product of two rows of Q - lambda I (rows of a rank-2 matrix span the
// plane normal to its null vector).  Sign convention: the component of largest magnitude is positive (first one
// on ties), the director being a headless vector.
#include "lq_internal.cuh"
#include "../../include/lq.h"

namespace {

constexpr int AB = 256;

__device__ __forceinline__ void cross3(const double a[3], const double b[3], double c[3]) {
    c[0] = a[1] * b[2] - a[2] * b[1];
    c[1] = a[2] * b[0] - a[0] * b[2];
    c[2] = a[0] * b[1] - a[1] * b[0];
}

__device__ __forceinline__ void top_eigenpair(double xx, double xy, double xz, double yy, double yz, double &lam,
                                              double n[3]) {
    const double zz = -xx - yy;
    const double p2 = xx * xx + yy * yy + zz * zz + 2.0 * (xy * xy + xz * xz + yz * yz);       // tr Q^2
    const double det = xx * (yy * zz - yz * yz) - xy * (xy * zz - yz * xz) + xz * (xy * yz - yy * xz);
    if (!(p2 > 0.0)) { lam = 0.0; n[0] = 0.0; n[1] = 0.0; n[2] = 1.0; return; }              // Q == 0: isotropic
    // lambda = 2 sqrt(p2/6) cos(phi/3), cos(phi) = det / (2 (p2/6)^{3/2}); the root with phi/3 in [0, pi/3] is the
    // largest.  The trigonometric part only seeds the iteration, so it runs in fp32 (relative error ~1e-6, nudged up
    // so that the seed sits on the convex side of the root); three fp64 Newton steps on
    // f(l) = l^3 - (p2/2) l - det then square the error each time (1e-6 -> 1e-12 -> rounding).
    const double s = sqrt(p2 / 6.0);
    const float rf = fminf(1.0f, fmaxf(-1.0f, (float)(det / (2.0 * s * s * s))));
    lam = 2.0 * s * (double)(__cosf(acosf(rf) * (1.0f / 3.0f)) * (1.0f + 3e-6f));
#pragma unroll
    for (int it = 0; it < 3; ++it) {
        const double f = (lam * lam - 0.5 * p2) * lam - det, fp = 3.0 * lam * lam - 0.5 * p2;
        if (fp > 0.0) lam -= f / fp;
    }
    const double r0[3] = {xx - lam, xy, xz}, r1[3] = {xy, yy - lam, yz}, r2[3] = {xz, yz, zz - lam};
    double c0[3], c1[3], c2[3];
    cross3(r0, r1, c0); cross3(r1, r2, c1); cross3(r2, r0, c2);
    const double d0 = c0[0] * c0[0] + c0[1] * c0[1] + c0[2] * c0[2], d1 = c1[0] * c1[0] + c1[1] * c1[1] + c1[2] * c1[2],
                 d2 = c2[0] * c2[0] + c2[1] * c2[1] + c2[2] * c2[2];
    double c[3] = {c0[0], c0[1], c0[2]};
    double d = d0;
    if (d1 > d) { c[0] = c1[0]; c[1] = c1[1]; c[2] = c1[2]; d = d1; }
    if (d2 > d) { c[0] = c2[0]; c[1] = c2[1]; c[2] = c2[2]; d = d2; }
    if (!(d > 0.0)) {                              // doubly degenerate top eigenvalue: any vector of the plane
        n[0] = 0.0; n[1] = 0.0; n[2] = 1.0;
        return;
    }
    const double inv = rsqrt(d);
    n[0] = c[0] * inv; n[1] = c[1] * inv; n[2] = c[2] * inv;
    const double a0 = fabs(n[0]), a1 = fabs(n[1]), a2 = fabs(n[2]);
    const double lead = (a0 >= a1 && a0 >= a2) ? n[0] : (a1 >= a2 ? n[1] : n[2]);
    if (lead < 0.0) { n[0] = -n[0]; n[1] = -n[1]; n[2] = -n[2]; }
}

__global__ void __launch_bounds__(AB) k_analyze(LqGeom g, const double *__restrict__ q, const uint8_t *__restrict__ flags,
                                                double thr, double *__restrict__ S, double *__restrict__ dir,
                                                uint8_t *__restrict__ defect, unsigned long long *__restrict__ count) {
    // dense (unpadded) outputs [N], [3][N], [N]; one row of x per block-row for coalesced stores
    const int x = blockIdx.x * blockDim.x + threadIdx.x;
    const int y = blockIdx.y, z = blockIdx.z;
    unsigned is_def = 0u;
    if (x < g.Lx) {
        const long long p = g.pidx(x, y, z), s = (long long)x + (long long)g.Lx * (y + (long long)g.Ly * z);
        const bool sim = !flags || (flags[p] & 3u) != 2u;
        double lam = 0.0, n[3] = {0.0, 0.0, 0.0};
        if (sim) {
            top_eigenpair(__ldcs(q + p), __ldcs(q + g.NP + p), __ldcs(q + 2 * g.NP + p), __ldcs(q + 3 * g.NP + p),
                          __ldcs(q + 4 * g.NP + p), lam, n);
            is_def = lam < thr ? 1u : 0u;
        }
        if (S) __stcs(S + s, lam);
        if (dir) { __stcs(dir + s, n[0]); __stcs(dir + g.N + s, n[1]); __stcs(dir + 2 * g.N + s, n[2]); }
        if (defect) defect[s] = (uint8_t)is_def;
    }
    const unsigned nd = __syncthreads_count(is_def);
    if (threadIdx.x == 0 && nd && count) atomicAdd(count, (unsigned long long)nd);
}

}  // namespace

void lq_launch_analyze(const LqGeom &g, const double *q, const uint8_t *flags, double thr, double *S, double *dir,
                       uint8_t *defect, unsigned long long *count, cudaStream_t st) {
    const int nt = g.Lx >= AB ? AB : (g.Lx + 31) / 32 * 32;      // one row of x per block-row
    dim3 grid((g.Lx + nt - 1) / nt, g.Ly, g.Lz);
    k_analyze<<<grid, nt, 0, st>>>(g, q, flags, thr, S, dir, defect, count);
}

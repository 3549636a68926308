// lq_descent.cu -- fixed-step gradient descent and Nesterov's accelerated gradient on the same force
// ("gradient descent (GD)", 289, 445 "Nesterov's accelerated gradient";
// readings DESIGN.md R23, R24):
//     y_k     = q_k                          (GD)
//     y_k     = q_k + mu (q_k - q_{k-1})     (Nesterov, q_{-1} = q_0)
//     q_{k+1} = y_k + eta F(y_k)             F = -dF/dq, simulated sites only
// ONE launch per step: the look-ahead point y is a pointwise function of (q_k, q_{k-1}), so every thread
// forms y at its own site and at the stencil neighbours it reads; nothing depends on another thread's output
// and the step needs no global scalar.  The same pass reduces |F|^2 and max|F_a|; the last block to finish
// sums the per-block partials in index order and sets the convergence flag on the device.
// Two kernels share the arithmetic:
//   k_descent       one thread per lattice site, general masked gather form (any constants, anchoring);
//   k_descent_sweep TMA-staged z-marching 7-point fast path for one-constant lattices (plain sites), with
//                   k_descent on the compacted list of non-plain sites when there are objects.
#include "lq_sweep.cuh"
#include "lq_sweep_dev.cuh"
#include "lq_site.cuh"
#include "../../include/lq.h"

#include <string>

namespace {
using namespace lqsw;

// y = q + mu (q - q_prev): the one expression every reader of y uses, so all copies round identically
__device__ __forceinline__ double lookahead(double q, double qp, double mu) { return __fma_rn(mu, q - qp, q); }

// accessor over the look-ahead field (lq_site.cuh's site_force reads tensors and flags through it)
template <bool NEST>
struct YAcc {
    const double *q, *qp;
    const uint8_t *flags;
    long long NP, sy, sz, p;
    double mu;
    __device__ __forceinline__ void Q(int dx, int dy, int dz, double o[6]) const {
        const long long i = p + dx + dy * sy + dz * sz;
#pragma unroll
        for (int c = 0; c < 5; ++c) {
            const double a = q[c * NP + i];
            o[c] = NEST ? lookahead(a, qp[c * NP + i], mu) : a;
        }
        o[5] = -o[0] - o[3];
    }
    __device__ __forceinline__ unsigned flag(int dx, int dy, int dz) const {
        return flags ? (unsigned)flags[p + dx + dy * sy + dz * sz] : 0xFCu;
    }
};

struct DescArgs {
    LqGeom g;
    LqPhys ph;
    LqFields f;
    const double *q, *qp;   // q_k, q_{k-1} (qp == q on the first step)
    double *qo;             // q_{k+1}
    double eta, mu, force_tol;
    const int *list;        // compacted site list (padded indices) or nullptr = every lattice site
    int n;                  // entries of list
    LqFireScalars *sc;      // step, FF, Fmax, converged live here
    double *partials;       // [2 * blocks] of this launch
    const double *extra;    // partials of a sweep launched before this kernel in the same step, or nullptr
    int n_extra;
    unsigned int *counter;
    int finish;             // this launch closes the step
};

constexpr int DB = 128;

// store one site of q_{k+1} and its periodic ghost images (width LQ_GH)
__device__ __forceinline__ void store_site(const LqGeom &g, double *qo, long long p, int x, int y, int z,
                                           const double o[5]) {
    const long long NP = g.NP;
#pragma unroll
    for (int c = 0; c < 5; ++c) qo[c * NP + p] = o[c];
    const int shx = ghost_shift(x, g.Lx, g.gwx), shy = ghost_shift(y, g.Ly, LQ_GH), shz = ghost_shift(z, g.Lz, LQ_GH);
    if (shx | shy | shz) {
        for (int m = 1; m < 8; ++m) {
            if (((m & 1) && !shx) || ((m & 2) && !shy) || ((m & 4) && !shz)) continue;
            const long long pg = p + ((m & 1) ? shx : 0) + ((m & 2) ? shy * g.sy : 0) + ((m & 4) ? shz * g.sz : 0);
#pragma unroll
            for (int c = 0; c < 5; ++c) qo[c * NP + pg] = o[c];
        }
    }
}


// Close a launch: block-reduce r = (|F|^2, max|F_a|), publish, and -- if this launch closes the step -- let the
// last block sum all partials in index order (bitwise reproducible) and advance (step, FF, Fmax, converged).
template <int NT>
__device__ __forceinline__ void finish_descent(const DescArgs &a, const double r[2], double *red, unsigned *s_last) {
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    constexpr int NW = NT / 32;
    const double w0 = warp_sum(r[0]), w1 = warp_max(r[1]);
    if (lane == 0) { red[wid] = w0; red[NW + wid] = w1; }
    __syncthreads();
    const unsigned nb = gridDim.x * gridDim.y * gridDim.z;
    const unsigned b = blockIdx.x + gridDim.x * (blockIdx.y + gridDim.y * blockIdx.z);
    if (tid == 0) {
        double t0 = red[0], t1 = red[NW];
        for (int w = 1; w < NW; ++w) { t0 += red[w]; t1 = fmax(t1, red[NW + w]); }
        a.partials[2 * b] = t0; a.partials[2 * b + 1] = t1;
        if (a.finish) {
            __threadfence();
            *s_last = atomicAdd(a.counter, 1u) == nb - 1 ? 1u : 0u;
        } else *s_last = 0u;
    }
    __syncthreads();
    if (!*s_last) return;
    __threadfence();
    double t0 = 0.0, t1 = 0.0;
    for (int i = tid; i < a.n_extra; i += NT) { t0 += __ldcg(a.extra + 2 * i); t1 = fmax(t1, __ldcg(a.extra + 2 * i + 1)); }
    for (unsigned i = tid; i < nb; i += NT) { t0 += __ldcg(a.partials + 2 * i); t1 = fmax(t1, __ldcg(a.partials + 2 * i + 1)); }
    t0 = warp_sum(t0); t1 = warp_max(t1);
    __syncthreads();
    if (lane == 0) { red[wid] = t0; red[NW + wid] = t1; }
    __syncthreads();
    if (tid == 0) {
        double FF = red[0], Fm = red[NW];
        for (int w = 1; w < NW; ++w) { FF += red[w]; Fm = fmax(Fm, red[NW + w]); }
        LqFireScalars nx = *a.sc;
        nx.step += 1; nx.FF = FF; nx.Fmax = Fm; nx.P = 0.0; nx.vv = 0.0;
        if (Fm < a.force_tol) nx.converged = 1;
        *a.sc = nx;
        *a.counter = 0u;
    }
}

// general form: one thread per site (of the whole lattice, or of a compacted list)
template <bool THREE, bool NEST>
__global__ void __launch_bounds__(DB) k_descent(const DescArgs a) {
    __shared__ double red[2 * (DB / 32)];
    __shared__ unsigned s_last;
    if (a.sc->converged) return;
    const long long i = (long long)blockIdx.x * DB + threadIdx.x;
    const long long NP = a.g.NP;
    double r[2] = {0.0, 0.0};
    const long long total = a.list ? (long long)a.n : a.g.N;
    if (i < total) {
        int x, y, z;
        long long p;
        if (a.list) {
            p = a.list[i];
            x = (int)(p % a.g.Px) - LQ_XO; y = (int)((p / a.g.Px) % a.g.Py) - LQ_GH; z = (int)(p / a.g.sz) - LQ_GH;
        } else {
            x = (int)(i % a.g.Lx); y = (int)((i / a.g.Lx) % a.g.Ly); z = (int)(i / ((long long)a.g.Lx * a.g.Ly));
            p = a.g.pidx(x, y, z);
        }
        const unsigned fl = a.f.flags ? a.f.flags[p] : 0xFCu;
        double o[5];
        if ((fl & 3u) != 2u) {
            int kind = 0; double W = 0.0, n[3] = {0.0, 0.0, 0.0};
            if (a.f.kind != nullptr && (fl & 3u) == 1u) {
                kind = a.f.kind[p];
                if (kind != 0) { W = a.f.W[p]; n[0] = a.f.axis[p]; n[1] = a.f.axis[NP + p]; n[2] = a.f.axis[2 * NP + p]; }
            }
            YAcc<NEST> acc{a.q, a.qp, a.f.flags, NP, a.g.sy, a.g.sz, p, a.mu};
            double F[5], Y[6];
            lqs::site_force<THREE>(a.ph, acc, fl, kind, W, n, F);
            acc.Q(0, 0, 0, Y);
#pragma unroll
            for (int c = 0; c < 5; ++c) {
                o[c] = __fma_rn(a.eta, F[c], Y[c]);
                r[0] = __fma_rn(F[c], F[c], r[0]);
                r[1] = fmax(r[1], fabs(F[c]));
            }
        } else {
#pragma unroll
            for (int c = 0; c < 5; ++c) o[c] = a.q[c * NP + p];      // object sites never move
        }
        store_site(a.g, a.qo, p, x, y, z, o);
    }
    finish_descent<DB>(a, r, red, &s_last);
}


// ---------------------------------------------------------------- one-constant fast path (plain sites)
// 7-point Laplacian with a fixed association and F of a pure-bulk one-constant site from its tensor and
// Laplacian (Eq. 5 + Eq. 11), explicit roundings.
__device__ __forceinline__ double lap7(double xl, double xr, double yu, double yd, double zm, double zp, double c) {
    return __fma_rn(-6.0, c, __dadd_rn(__dadd_rn(__dadd_rn(xl, xr), __dadd_rn(yu, yd)), __dadd_rn(zm, zp)));
}
__device__ __forceinline__ void force1(const LqPhys &ph, const double q[5], const double lap[5], double F[5]) {
    const double a = q[0], b = q[1], c = q[2], d = q[3], e = q[4], f = -(a + d);
    const double aa = a * a, bb = b * b, cc = c * c, dd = d * d, ee = e * e, ff = f * f;
    const double tr = __dadd_rn(__dadd_rn(__dadd_rn(aa, dd), ff), 2.0 * __dadd_rn(__dadd_rn(bb, cc), ee));
    const double k = __fma_rn(ph.C, tr, ph.A);
    const double bf = __dadd_rn(bb, -ff);
    const double dxx = __dadd_rn(__dadd_rn(aa, -ee), bf);          // (Q^2)xx - (Q^2)zz
    const double dyy = __dadd_rn(__dadd_rn(dd, -cc), bf);          // (Q^2)yy - (Q^2)zz
    const double qxy = __fma_rn(c, e, __fma_rn(b, d, a * b));
    const double qxz = __fma_rn(c, f, __fma_rn(b, e, a * c));
    const double qyz = __fma_rn(e, f, __fma_rn(d, e, b * c));
    const double L1 = ph.L1, L2x = 2.0 * ph.L1, mB = -ph.B, m2B = -2.0 * ph.B, m2k = -2.0 * k;
    // Gxx - Gzz = k (a - f) + B dxx with a - f = 2a + d
    // + Fx: constant external-field force (Eq. 13), folded into the FMAs
    F[0] = __fma_rn(L1, __fma_rn(2.0, lap[0], lap[3]), __fma_rn(mB, dxx, __fma_rn(-k, __fma_rn(2.0, a, d), ph.Fx[0])));
    F[3] = __fma_rn(L1, __fma_rn(2.0, lap[3], lap[0]), __fma_rn(mB, dyy, __fma_rn(-k, __fma_rn(2.0, d, a), ph.Fx[3])));
    F[1] = __fma_rn(L2x, lap[1], __fma_rn(m2B, qxy, __fma_rn(m2k, b, ph.Fx[1])));
    F[2] = __fma_rn(L2x, lap[2], __fma_rn(m2B, qxz, __fma_rn(m2k, c, ph.Fx[2])));
    F[4] = __fma_rn(L2x, lap[4], __fma_rn(m2B, qyz, __fma_rn(m2k, e, ph.Fx[4])));
}

// CTA = 32 x 16 columns marching a z-chunk.  Per plane one elected thread issues one (GD) or two (Nesterov)
// 4-D TMA boxes (36 x 18 x 1 x 5: tile + 1 halo; the innermost start coordinate must be 16-byte aligned, hence
// x0-2) into an NS-slot mbarrier ring.  A thread keeps the look-ahead column y(z-1), y(z), y(z+1) of its site in
// registers and reads the four in-plane neighbours from the landed boxes; y is formed on the fly.
template <bool NEST, int NS_, int TY_ = 16>
struct DS {
    static constexpr int TX = 32, TY = TY_, NT = TX * TY, NS = NS_;
    static constexpr int SW = TX + 4, SH = TY + 2, SPLANE = SW * SH;
    static constexpr int BOX_BYTES = 5 * SPLANE * 8, BOX_STRIDE = (BOX_BYTES + 127) / 128 * 128;
    static constexpr int NF = NEST ? 2 : 1;
    static constexpr int SLOT = NF * BOX_STRIDE;
    static constexpr int OFF_BAR = NS * SLOT;
    static constexpr int OFF_RED = OFF_BAR + 8 * NS_ + (8 * NS_ % 16);
    static constexpr int SMEM_BYTES = OFF_RED + 2 * (NT / 32) * 8 + 16;
};

// THREE: L2/L3 != 0 -- the 19-point constant-weight stencil (lqs::bulk_force_threeconst) reads planes k-1, k, k+1
// from the ring (three live slots instead of two).
// XT: extra distortion terms in the 19-point stencil (bit 0 chiral L4, bit 1 cubic L6)
// The cubic-term (L6) instantiations run 32 x 8 tiles of 256 threads: their 19-point cubic stencil needs the
// 255-register budget (at 128 registers it spilled ~800 B per thread).
template <bool NEST, bool MASKED, bool THREE, int XT, int NS>
__global__ void __launch_bounds__(((XT & 2) ? 8 : 16) * 32, 1)
k_descent_sweep(const __grid_constant__ CUtensorMap tq, const __grid_constant__ CUtensorMap tp, const DescArgs a,
                const uint8_t *__restrict__ plain, const uint32_t *__restrict__ bond, int zc) {
    // masked lattices: with one elastic constant every simulated site is handled here from its bond code
    // (lq_internal.cuh LQ_BOND_*: six weights of the boundary-aware 7-point stencil, + object / anchoring
    // bits; the same codes the FIRE recompute sweep uses); with three constants `plain` marks the sites of the
    // constant-weight 19-point stencil and the rest goes to k_descent on the non-plain list
    constexpr bool BOND = MASKED && !THREE;
    using C = DS<NEST, NS, (XT & 2) ? 8 : 16>;
    extern __shared__ __align__(1024) unsigned char smem[];
    __shared__ unsigned s_last;
    if (a.sc->converged) return;
    uint64_t *full = reinterpret_cast<uint64_t *>(smem + C::OFF_BAR);
    double *red = reinterpret_cast<double *>(smem + C::OFF_RED);
    const int tid = threadIdx.x, tx = tid & 31, ty = tid >> 5;
    const int x0 = blockIdx.x * C::TX, y0 = blockIdx.y * C::TY;
    const int zb = blockIdx.z * zc, ze = min(a.g.Lz, zb + zc);
    const int x = x0 + tx, y = y0 + ty;
    const bool active = x < a.g.Lx && y < a.g.Ly;
    const int nplanes = ze - zb + 2;              // planes zb-1 .. ze
    const double mu = a.mu, eta = a.eta;

    if (tid == 0) {
#pragma unroll
        for (int i = 0; i < NS; ++i) mbar_init(&full[i], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    auto issue = [&](int j, int s) {               // plane zb-1+j -> slot s
        unsigned char *dst = smem + s * C::SLOT;
        const int cx = x0 + LQ_XO - 2, cy = y0 + LQ_GH - 1, cz = zb - 1 + j + LQ_GH;
        mbar_expect_tx(&full[s], (uint32_t)(C::NF * C::BOX_BYTES));
        tma_load_4d(dst, &tq, &full[s], cx, cy, cz, 0);
        if (NEST) tma_load_4d(dst + C::BOX_STRIDE, &tp, &full[s], cx, cy, cz, 0);
    };
    if (tid == 0)
        for (int j = 0; j < NS && j < nplanes; ++j) issue(j, j);

    const int sidx = (ty + 1) * C::SW + tx + 2;    // own site in a staged box
    auto Y = [&](const double *sq, int c, int off) -> double {
        const double v = sq[c * C::SPLANE + sidx + off];
        return NEST ? lookahead(v, sq[C::BOX_STRIDE / 8 + c * C::SPLANE + sidx + off], mu) : v;
    };
    double ym[5], yc[5], r[2] = {0.0, 0.0};
#pragma unroll
    for (int c = 0; c < 5; ++c) ym[c] = yc[c] = 0.0;
    long long p = a.g.pidx(x, y, zb - 1);          // padded index of the plane handled now (k = zb + j - 2)
    unsigned pb_next = BOND ? LQ_BOND_PLAIN : 1u;
    int s0 = 0, s1 = NS - 1, s2 = NS - 2;        // ring slots of planes j, j-1, j-2
    uint32_t par = 0;
    for (int j = 0; j < nplanes; ++j) {
        const unsigned pb = pb_next;
        pb_next = BOND ? LQ_BOND_PLAIN : 1u;
        if (MASKED && active && j >= 1 && j + 1 < nplanes) pb_next = BOND ? bond[p + a.g.sz] : (unsigned)plain[p + a.g.sz];
        mbar_wait(&full[s0], par);
        const double *sj = reinterpret_cast<const double *>(smem + s0 * C::SLOT);
        double yn[5];
#pragma unroll
        for (int c = 0; c < 5; ++c) yn[c] = Y(sj, c, 0);
        if (j >= 2 && active) {
            const int k = zb + j - 2;
            const double *sb = reinterpret_cast<const double *>(smem + s1 * C::SLOT);
            if (BOND && pb != LQ_BOND_PLAIN) {
                if (pb & LQ_BOND_OBJECT) store_site(a.g, a.qo, p, x, y, k, yc);     // object site: y == q, never moves
                else {
                    const double w0 = lq_bond_weight(pb, 0), w1 = lq_bond_weight(pb, 1), w2 = lq_bond_weight(pb, 2),
                                 w3 = lq_bond_weight(pb, 3), w4 = lq_bond_weight(pb, 4), w5 = lq_bond_weight(pb, 5);
                    double lap[5], F[5], o[5];
#pragma unroll
                    for (int c = 0; c < 5; ++c) {
                        const double qx = yc[c];
                        lap[c] = (w0 * (Y(sb, c, 1) - qx) + w1 * (Y(sb, c, -1) - qx)) +
                                 (w2 * (Y(sb, c, C::SW) - qx) + w3 * (Y(sb, c, -C::SW) - qx)) +
                                 (w4 * (yn[c] - qx) + w5 * (ym[c] - qx));
                    }
                    force1(a.ph, yc, lap, F);
                    if (pb & LQ_BOND_ANCH) {          // Eq. 14 / 15 at a boundary site with an anchoring record
                        const int kind = a.f.kind[p];
                        if (kind != 0) {
                            const long long NP = a.g.NP;
                            const double n[3] = {a.f.axis[p], a.f.axis[NP + p], a.f.axis[2 * NP + p]};
                            const double Q[6] = {yc[0], yc[1], yc[2], yc[3], yc[4], -yc[0] - yc[3]};
                            double G[3][3] = {{0.0, 0.0, 0.0}, {0.0, 0.0, 0.0}, {0.0, 0.0, 0.0}}, Fa[5];
                            lqs::anchoring(a.ph, kind, a.f.W[p], n, Q, G);
                            lqs::G_to_F(G, Fa);
#pragma unroll
                            for (int c = 0; c < 5; ++c) F[c] += Fa[c];
                        }
                    }
#pragma unroll
                    for (int c = 0; c < 5; ++c) {
                        o[c] = __fma_rn(eta, F[c], yc[c]);
                        r[0] = __fma_rn(F[c], F[c], r[0]);
                        r[1] = fmax(r[1], fabs(F[c]));
                    }
                    store_site(a.g, a.qo, p, x, y, k, o);
                }
            } else if (!MASKED || BOND || pb == 1u) {
                double F[5], o[5];
                if (!THREE) {
                    double lap[5];
#pragma unroll
                    for (int c = 0; c < 5; ++c)
                        lap[c] = lap7(Y(sb, c, -1), Y(sb, c, 1), Y(sb, c, -C::SW), Y(sb, c, C::SW), ym[c], yn[c], yc[c]);
                    force1(a.ph, yc, lap, F);
                } else {
                    const double *sa = reinterpret_cast<const double *>(smem + s2 * C::SLOT);
                    auto get = [&](int c, int dx, int dy, int dz) -> double {
                        if (dz != 0 && dx == 0 && dy == 0) return dz < 0 ? ym[c] : yn[c];
                        return Y(dz < 0 ? sa : (dz > 0 ? sj : sb), c, dy * C::SW + dx);
                    };
                    lqs::bulk_force_threeconst<(XT & 1) != 0, (XT & 2) != 0>(a.ph, get, yc, F);
                }
#pragma unroll
                for (int c = 0; c < 5; ++c) {
                    o[c] = __fma_rn(eta, F[c], yc[c]);
                    r[0] = __fma_rn(F[c], F[c], r[0]);
                    r[1] = fmax(r[1], fabs(F[c]));
                }
                store_site(a.g, a.qo, p, x, y, k, o);
            } else if (pb == 2u) {
                store_site(a.g, a.qo, p, x, y, k, yc);     // object site: y == q, never moves
            }                                              // pb == 0: left to k_descent on the non-plain list
        }
        if (j >= 1) p += a.g.sz;
#pragma unroll
        for (int c = 0; c < 5; ++c) { ym[c] = yc[c]; yc[c] = yn[c]; }
        // the oldest live plane (j-1, or j-2 for the 19-point stencil) has been read by every thread: refill its slot
        __syncthreads();
        constexpr int DEAD = THREE ? 2 : 1;
        if (tid == 0 && j >= DEAD && j - DEAD + NS < nplanes) issue(j - DEAD + NS, THREE ? s2 : s1);
        s2 = s1;
        s1 = s0;
        if (++s0 == NS) { s0 = 0; par ^= 1u; }
    }
    finish_descent<C::NT>(a, r, red, &s_last);
}

}  // namespace

struct LqDescentPlan {
    double *partials = nullptr;       // k_descent blocks
    size_t cap = 0;
    double *sweep_partials = nullptr; // k_descent_sweep CTAs
    size_t sweep_cap = 0;
    unsigned int *counter = nullptr;
    // one-constant fast path
    CUtensorMap map[3];
    double *mapped[3] = {nullptr, nullptr, nullptr};
    int map_ty = 0;                   // tile rows the maps' boxes were made for
    uint8_t *plain = nullptr;         // per-site plain byte (masked lattices, three constants)
    uint32_t *bond = nullptr;         // per-site bond code (masked lattices, one constant)
    bool bond_built = false, list_built = false;
    int *list = nullptr;              // index-ordered non-plain simulated sites
    int n_list = 0;
    const uint8_t *flags_seen = nullptr;
    bool sites_dirty = true;
    bool attr_set[32] = {};
};

void lq_descent_destroy(LqDescentPlan *p) {
    if (!p) return;
    cudaFree(p->partials);
    cudaFree(p->sweep_partials);
    cudaFree(p->counter);
    cudaFree(p->plain);
    cudaFree(p->bond);
    cudaFree(p->list);
    delete p;
}
void lq_descent_invalidate(LqDescentPlan *p) {
    if (p) p->sites_dirty = true;
}

namespace {
constexpr int NS_GD = 6, NS_NEST = 4;   // ring depth: 6 x 25.4 KB (GD), 4 x 50.8 KB (Nesterov)

template <bool NEST, bool MASKED, bool THREE, int XT = 0>
cudaError_t launch_sweep_t(LqDescentPlan *pl, dim3 grid, const CUtensorMap &mq, const CUtensorMap &mp, const DescArgs &a,
                           int zc, cudaStream_t st) {
    constexpr int NS = NEST ? NS_NEST : NS_GD;
    using C = DS<NEST, NS, (XT & 2) ? 8 : 16>;
    const int v = 8 * XT + (THREE ? 4 : 0) + (NEST ? 2 : 0) + (MASKED ? 1 : 0);
    if (!pl->attr_set[v]) {
        cudaError_t e = cudaFuncSetAttribute(k_descent_sweep<NEST, MASKED, THREE, XT, NS>,
                                             cudaFuncAttributeMaxDynamicSharedMemorySize, C::SMEM_BYTES);
        if (e != cudaSuccess) return e;
        pl->attr_set[v] = true;
    }
    k_descent_sweep<NEST, MASKED, THREE, XT, NS><<<grid, C::NT, C::SMEM_BYTES, st>>>(mq, mp, a, pl->plain, pl->bond, zc);
    return cudaGetLastError();
}
template <bool NEST, bool MASKED>
cudaError_t launch_sweep(bool three, LqDescentPlan *pl, dim3 grid, const CUtensorMap &mq, const CUtensorMap &mp,
                         const DescArgs &a, int zc, cudaStream_t st) {
    const int xt = (a.ph.L4 != 0.0 ? 1 : 0) | (a.ph.L6 != 0.0 ? 2 : 0);
    if (three && xt == 1) return launch_sweep_t<NEST, MASKED, true, 1>(pl, grid, mq, mp, a, zc, st);
    if (three && xt == 2) return launch_sweep_t<NEST, MASKED, true, 2>(pl, grid, mq, mp, a, zc, st);
    if (three && xt == 3) return launch_sweep_t<NEST, MASKED, true, 3>(pl, grid, mq, mp, a, zc, st);
    return three ? launch_sweep_t<NEST, MASKED, true>(pl, grid, mq, mp, a, zc, st)
                 : launch_sweep_t<NEST, MASKED, false>(pl, grid, mq, mp, a, zc, st);
}
}  // namespace

// Runs up to max_steps steps.  buf[0] holds q_0 with a valid ghost shell; nbuf = 2 (GD) or 3 (Nesterov) rotating
// buffers.  On return *final is the index of the buffer that holds the last iterate and *h the scalars.
// path: 0 = fast path where it applies (one-constant: TMA sweep over plain sites + k_descent on the non-plain
// list), 1 = k_descent over every site.
int lq_descent_run(LqDescentPlan **planp, int method, int path, const LqGeom &g, const LqPhys &ph, const LqFields &f,
                   double *const *buf, int nbuf, int *final, LqFireScalars *dsc, double eta, double mu,
                   double force_tol, long max_steps, cudaStream_t st, long *launches, long *sweeps,
                   LqFireScalars *h, std::string &err) {
    LqDescentPlan *pl = *planp;
    if (!pl) { pl = new LqDescentPlan(); *planp = pl; }
    const bool three = lq_three(ph);
    const bool nest = method == LQ_MIN_NESTEROV;
    const bool masked = f.flags != nullptr;
    const bool fast = path == 0;
    cudaError_t e;
#define DESC_CUDA(call) do { e = (call); if (e != cudaSuccess) { err = std::string("lq_descent: ") + cudaGetErrorString(e); return LQ_ERR_CUDA; } } while (0)

    // fast path set-up: tensor maps of the rotating buffers, z-chunking, plain map + non-plain list
    dim3 grid(1, 1, 1);
    int zc = g.Lz;
    if (fast) {
        const int TY = (three && ph.L6 != 0.0) ? 8 : 16;       // tile rows: see k_descent_sweep
        for (int i = 0; i < nbuf; ++i)
            if (pl->mapped[i] != buf[i] || pl->map_ty != TY) {
                if (!lq_make_box_map(&pl->map[i], g, buf[i], 36, TY + 2)) { err = "lq_descent: cuTensorMapEncodeTiled failed"; return LQ_ERR_CUDA; }
                pl->mapped[i] = buf[i];
            }
        pl->map_ty = TY;
        const int ntx = (g.Lx + 31) / 32, nty = (g.Ly + TY - 1) / TY;
        long long best = -1;
        for (int nzc = 1; nzc <= (g.Lz + 3) / 4; ++nzc) {          // equal chunks, modelled makespan on 148 SMs
            const int c = (g.Lz + nzc - 1) / nzc;
            const long long ncta = (long long)ntx * nty * ((g.Lz + c - 1) / c);
            const long long cost = ((ncta + 147) / 148) * (c + (three ? 5 : 4));
            if (best < 0 || cost < best) { best = cost; zc = c; }
        }
        grid = dim3(ntx, nty, (g.Lz + zc - 1) / zc);
        const size_t ncta = (size_t)grid.x * grid.y * grid.z;
        if (pl->sweep_cap < 2 * ncta) {
            cudaFree(pl->sweep_partials); pl->sweep_partials = nullptr; pl->sweep_cap = 0;
            if (cudaMalloc(&pl->sweep_partials, 2 * ncta * sizeof(double)) != cudaSuccess) { err = "lq_descent: cudaMalloc failed"; return LQ_ERR_NOMEM; }
            pl->sweep_cap = 2 * ncta;
        }
        if (masked && (pl->sites_dirty || pl->flags_seen != f.flags)) { pl->bond_built = pl->list_built = false; }
        if (masked && !three && !pl->bond_built) {
            // one constant: bond codes, every simulated site in the sweep (no second kernel)
            if (!pl->bond && cudaMalloc(&pl->bond, (size_t)g.NP * sizeof(uint32_t)) != cudaSuccess) { err = "lq_descent: cudaMalloc failed"; return LQ_ERR_NOMEM; }
            DESC_CUDA(cudaMemsetAsync(pl->bond, 0, (size_t)g.NP * sizeof(uint32_t), st));
            lq_launch_bond_map(g, f.flags, f.kind, pl->bond, st);
            *launches += 1;
            pl->bond_built = true;
        }
        if (masked && three && !pl->list_built) {
            if (!pl->plain && cudaMalloc(&pl->plain, (size_t)g.NP) != cudaSuccess) { err = "lq_descent: cudaMalloc failed"; return LQ_ERR_NOMEM; }
            DESC_CUDA(cudaMemsetAsync(pl->plain, 0, (size_t)g.NP, st));
            lq_launch_plain_map(g, f.flags, pl->plain, st);
            *launches += 1;
            if (lq_fixup_build_list(g, f.flags, pl->plain, &pl->list, &pl->n_list, st) != 0) { err = "lq_descent: building the non-plain site list failed"; return LQ_ERR_NOMEM; }
            pl->list_built = true;
        }
        if (masked) { pl->sites_dirty = false; pl->flags_seen = f.flags; }
    }
    const long long nsites = fast ? ((masked && three) ? pl->n_list : 0) : g.N;
    const unsigned nblk = (unsigned)((nsites + DB - 1) / DB);
    if (pl->cap < (size_t)2 * nblk) {
        cudaFree(pl->partials); pl->partials = nullptr; pl->cap = 0;
        if (cudaMalloc(&pl->partials, (size_t)2 * nblk * sizeof(double)) != cudaSuccess) { err = "lq_descent: cudaMalloc failed"; return LQ_ERR_NOMEM; }
        pl->cap = (size_t)2 * nblk;
    }
    if (!pl->counter && cudaMalloc(&pl->counter, sizeof(unsigned int)) != cudaSuccess) { err = "lq_descent: cudaMalloc failed"; return LQ_ERR_NOMEM; }
    DESC_CUDA(cudaMemsetAsync(pl->counter, 0, sizeof(unsigned int), st));

    DescArgs a;
    a.g = g; a.ph = ph; a.f = f; a.eta = eta; a.mu = nest ? mu : 0.0; a.force_tol = force_tol;
    a.sc = dsc; a.counter = pl->counter;
    const bool second = nblk > 0;                  // a k_descent launch closes the step
    const int per_step = (fast ? 1 : 0) + (second ? 1 : 0);
    const long chunk = force_tol > 0.0 ? 100 : (1L << 30);
    long done = 0;
    while (done < max_steps) {
        const long n = (max_steps - done) < chunk ? (max_steps - done) : chunk;
        for (long i = 0; i < n; ++i) {
            const long k = done + i;
            const int in = (int)(k % nbuf), out = (int)((k + 1) % nbuf), prev = k == 0 ? in : (int)((k - 1) % nbuf);
            a.q = buf[in]; a.qp = buf[prev]; a.qo = buf[out];
            if (fast) {
                a.list = nullptr; a.n = 0; a.partials = pl->sweep_partials; a.extra = nullptr; a.n_extra = 0;
                a.finish = second ? 0 : 1;
                if (nest) e = masked ? launch_sweep<true, true>(three, pl, grid, pl->map[in], pl->map[prev], a, zc, st)
                                     : launch_sweep<true, false>(three, pl, grid, pl->map[in], pl->map[prev], a, zc, st);
                else e = masked ? launch_sweep<false, true>(three, pl, grid, pl->map[in], pl->map[in], a, zc, st)
                                : launch_sweep<false, false>(three, pl, grid, pl->map[in], pl->map[in], a, zc, st);
                DESC_CUDA(e);
            }
            if (second) {
                a.list = fast ? pl->list : nullptr; a.n = fast ? pl->n_list : 0; a.partials = pl->partials;
                a.extra = fast ? pl->sweep_partials : nullptr; a.n_extra = fast ? (int)(grid.x * grid.y * grid.z) : 0;
                a.finish = 1;
                if (three) {
                    if (nest) k_descent<true, true><<<nblk, DB, 0, st>>>(a);
                    else k_descent<true, false><<<nblk, DB, 0, st>>>(a);
                } else {
                    if (nest) k_descent<false, true><<<nblk, DB, 0, st>>>(a);
                    else k_descent<false, false><<<nblk, DB, 0, st>>>(a);
                }
                DESC_CUDA(cudaGetLastError());
            }
        }
        done += n;
        *launches += per_step * n;
        *sweeps += n;
        if (force_tol > 0.0) {
            DESC_CUDA(cudaMemcpyAsync(h, dsc, sizeof(*h), cudaMemcpyDeviceToHost, st));
            DESC_CUDA(cudaStreamSynchronize(st));
            if (h->converged) break;
        }
    }
    DESC_CUDA(cudaMemcpyAsync(h, dsc, sizeof(*h), cudaMemcpyDeviceToHost, st));
    DESC_CUDA(cudaStreamSynchronize(st));
#undef DESC_CUDA
    *final = (int)(h->step % nbuf);
    return LQ_OK;
}

// lq_sweep_rc.cu -- one-constant hot path with the force RECOMPUTED instead of stored (sm_100a).
//
// State carried between FIRE steps is only (q, vc): 4 x 5 fp64 per site-update = 160 B of compulsory
// HBM traffic; the force at q, needed for the lazy velocity rescale and the first half
// kick, is re-evaluated from q on the tile plus a one-site halo.  Per step and site
// (Algorithm 1):
//     F   = force(q)                               on tile + 1 halo   (needs q on tile + 2 halo)
//     v_k = mix_a vc + (mix_b + dt/2) F ; q' = q + dt v_k             on tile + 1 halo
//     F'  = force(q') ; vc' = v_k + dt/2 F' ; partial sums            on the tile
// Tiling: CTA = 32 x 16 columns marching over a z-range taken from a work table (longest items first, so the
// hardware's in-order CTA dispatch is a longest-processing-time schedule).  Per plane one elected thread issues
// two 4-D TMA boxes: q (36 x 20 x 1 x 5, start x0-2: the innermost start coordinate must be 16-byte aligned) into a
// 4-slot ring that doubles as the z-window of the first stencil, and vc (36 x 18 x 1 x 5) into a 2-slot
// stage; q' planes live in a 2-slot shared-memory ring and, for the thread's own column, in registers.
//
// Masked lattices (MASKED): EVERY simulated site is handled here -- no second kernel.  With one elastic constant
// the boundary-aware force (gather form) is a 7-point stencil whose six bond
// weights a^s_k(x) [w_k(x) + w_k(x + s k)] take the values 0, 1, 3/2, 2; they come from a per-site bond
// code built once per lq_set_sites.  Sites whose code says 'all weights 1' run the same instruction sequence as
// the unmasked kernel (so every CTA that evaluates such a site, as its own or as a halo copy, gets the same
// bits); the anchoring terms of Eq. 14 / 15 are added at boundary sites from their
// (kind, W, axis) record.
//
// FIRST: the first sweep of a lq_fire_minimize call.  Its phase 1 evaluates F(q_0) anyway; it also reduces
// |F(q_0)|^2 and max|F_a(q_0)|, which is the stop test of Algorithm 1's initialisation -- no separate force pass.
#include "lq_sweep.cuh"
#include "lq_sweep_dev.cuh"
#include "lq_site.cuh"

#include <type_traits>

namespace {
using namespace lqsw;

struct RC {
    static constexpr int TX = 32, TY = 16, NT = TX * TY;
    static constexpr int RW = TX + 4, RH = TY + 4, RPLANE = RW * RH;          // raw q box (tile + 2 halo)
    static constexpr int VW = TX + 4, VH = TY + 2, VPLANE = VW * VH;          // vc box (x0-2.., y0-1..)
    static constexpr int BXW = TX + 2, BYH = TY + 2, PLANE = BXW * BYH;       // q' ring (tile + 1 halo)
    static constexpr int Q_BYTES = 5 * RPLANE * 8, Q_STRIDE = (Q_BYTES + 127) / 128 * 128;
    static constexpr int V_BYTES = 5 * VPLANE * 8, V_STRIDE = (V_BYTES + 127) / 128 * 128;
    static constexpr int N_STRIDE = (5 * PLANE * 8 + 127) / 128 * 128;
    static constexpr int NQ = 4, NV = 2, NN = 2;
    static constexpr int OFF_V = NQ * Q_STRIDE;
    static constexpr int OFF_N = OFF_V + NV * V_STRIDE;
    static constexpr int OFF_BAR = OFF_N + NN * N_STRIDE;
    static constexpr int OFF_RED = OFF_BAR + 64;
    static constexpr int OFF_TS = OFF_RED + 4 * (NT / 32) * 8;     // tile summaries of this CTA's planes
    static constexpr int MAXZC = 126;                              // ts[] holds ze - zb + 2 <= 128 entries
    static constexpr int OFF_CODE = OFF_TS + 128;                  // bond codes: 4 slots x (NT own + 128 halo) x u32
    static constexpr int SMEM_BYTES = OFF_CODE + 4 * (NT + 128) * 4;
};
static_assert(RC::SMEM_BYTES <= 232448, "shared memory budget");

// Anchoring force of one boundary site, added to F (Eq. 14 / 15; lqs::anchoring).  Under a rare
// branch: it runs on the few per cent of sites next to objects (inlined: ptxas fits it in the 128-register budget without spills; an out-of-line call spilled the loop-carried columns).
struct F5 { double a, b, c, d, e; };
__device__ __forceinline__ F5 anchor_force(const LqPhys &ph, const LqFields &f, long long NP, long long p, double qxx,
                                        double qxy, double qxz, double qyy, double qyz) {
    F5 o = {0.0, 0.0, 0.0, 0.0, 0.0};
    const int kind = f.kind[p];
    if (kind == 0) return o;
    const double W = f.W[p];
    const double n[3] = {f.axis[p], f.axis[NP + p], f.axis[2 * NP + p]};
    const double Q[6] = {qxx, qxy, qxz, qyy, qyz, -qxx - qyy};
    double G[3][3] = {{0.0, 0.0, 0.0}, {0.0, 0.0, 0.0}, {0.0, 0.0, 0.0}};
    lqs::anchoring(ph, kind, W, n, Q, G);
    double Fa[5];
    lqs::G_to_F(G, Fa);
    o.a = Fa[0]; o.b = Fa[1]; o.c = Fa[2]; o.d = Fa[3]; o.e = Fa[4];
    return o;
}

template <bool MASKED, bool FIRST>
__global__ void __launch_bounds__(RC::NT, 1)
k_sweep_rc(const __grid_constant__ CUtensorMap tq, const __grid_constant__ CUtensorMap tv, const SweepArgs a) {
    extern __shared__ __align__(1024) unsigned char smem[];
    const LqFireScalars sc = *a.sc;
    if (sc.converged) return;

    uint64_t *full = reinterpret_cast<uint64_t *>(smem + RC::OFF_BAR);   // [NQ]
    double *red = reinterpret_cast<double *>(smem + RC::OFF_RED);
    const int tid = threadIdx.x;
    const int tx = tid % RC::TX, ty = tid / RC::TX;
    const int4 wk = a.work[blockIdx.x];
    const int bx = wk.x, by = wk.y;
    const int x0 = bx * RC::TX, y0 = by * RC::TY;
    const int zb = wk.z, ze = wk.w;
    const int x = x0 + tx, y = y0 + ty;
    const bool active = x < a.g.Lx && y < a.g.Ly;
    const int nplanes = ze - zb + 4;              // raw q planes zb-2 .. ze+1
    const long long NP = a.g.NP;

    if (tid == 0) {
#pragma unroll
        for (int i = 0; i < RC::NQ; ++i) mbar_init(&full[i], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    uint8_t *ts = smem + RC::OFF_TS;              // ts[i] = summary of plane zb-1+i
    if (MASKED && tid < ze - zb + 2)
        ts[tid] = a.tsum[((size_t)(zb + tid) * a.nty + by) * a.ntx + bx];
    __syncthreads();

    // issue(j): raw q plane zb-2+j -> q slot j%4; with it (j >= 2) vc plane zb-3+j -> v slot (j-1)%2
    auto issue = [&](int j) {
        const int s = j & 3;
        const int cx = x0 + LQ_XO - 2;
        const bool withv = j >= 2;
        mbar_expect_tx(&full[s], (uint32_t)RC::Q_BYTES + (withv ? (uint32_t)RC::V_BYTES : 0u));
        tma_load_4d(smem + s * RC::Q_STRIDE, &tq, &full[s], cx, y0 + LQ_GH - 2, zb - 2 + j + LQ_GH, 0);
        if (withv)
            tma_load_4d(smem + RC::OFF_V + ((j - 1) & 1) * RC::V_STRIDE, &tv, &full[s], cx, y0 + LQ_GH - 1,
                        zb - 3 + j + LQ_GH, 0);
    };
    if (tid == 0)
        for (int j = 0; j < 4 && j < nplanes; ++j) issue(j);

    const LqStepCoef kc = lq_step_coef(sc, a.fc);
    const double dt = kc.dt, ma = kc.ma, cF = kc.cF, hdt = kc.kick;
    double qm[5], qc[5], qp[5], vk0[5], vk1[5];
#pragma unroll
    for (int c = 0; c < 5; ++c) qm[c] = qc[c] = qp[c] = vk0[c] = vk1[c] = 0.0;
    double r[4] = {0.0, 0.0, 0.0, 0.0};
    double r0[2] = {0.0, 0.0};

    // halo share: perimeter cell (hx, hy) of the 34 x 18 q' box; own cell is (tx+1, ty+1).  The 100 perimeter cells
    // go to the first four warps, 25 lanes each: 8 side cells (4 consecutive rows, left and right) + 17 cells of the
    // top / bottom rows.  A column of the 36-wide TMA box strides 72 banks = 8 (mod 32), so rows 4 apart collide:
    // with at most one row of each residue per warp the side cells' shared-memory accesses are conflict-free among
    // themselves (all 32 side cells in one warp, as before, made every one of its accesses 4-way conflicted).
    int hx = -1, hy = -1;
    if (tid < 128) {
        const int w = tid >> 5, l = tid & 31;
        if (l < 8) { hy = 1 + 4 * w + (l >> 1); hx = (l & 1) ? RC::BXW - 1 : 0; }
        else if (l < 25) {
            const int t = 17 * w + (l - 8);                  // 0 .. 67: top row, then bottom row
            if (t < RC::BXW) { hx = t; hy = 0; }
            else { hx = t - RC::BXW; hy = RC::BYH - 1; }
        }
    }
    static_assert(RC::TY == 16 && 4 * 17 == 2 * RC::BXW, "halo mapping assumes a 32 x 16 tile");

    // Bond codes (masked lattices) of the own cell and the halo cell: cp.async'd into shared memory one plane ahead,
    // and only for planes whose tile + halo holds a non-plain site, so that (i) no dependent global load gates a
    // plane and (ii) they cost the plane loop no registers.  Planes whose tile + halo is all plain (the tile
    // summary says so; the bulk of any lattice with walls or colloids) run body<false>: the very instruction
    // sequence of the unmasked kernel.
    const bool own_in = x <= a.g.Lx && y <= a.g.Ly;
    const bool halo_in = hx >= 0 && x0 - 1 + hx <= a.g.Lx && y0 - 1 + hy <= a.g.Ly;
    uint32_t *cown = reinterpret_cast<uint32_t *>(smem + RC::OFF_CODE) + tid;                    // [4][NT]
    uint32_t *chalo = reinterpret_cast<uint32_t *>(smem + RC::OFF_CODE) + 4 * RC::NT + tid;      // [4][NHALO pad 128]

    // one iteration of the plane loop; GEN = the general (masked) form, evaluated per site from its bond code
    auto body = [&](auto gen_tag, int j) {
        constexpr bool GEN = decltype(gen_tag)::value;
        const int zc = zb + j - 3;                 // plane whose q' is produced now (zb-1 .. ze)
        const double *ra = reinterpret_cast<const double *>(smem + ((j - 2) & 3) * RC::Q_STRIDE);   // raw z-1
        const double *rb = reinterpret_cast<const double *>(smem + ((j - 1) & 3) * RC::Q_STRIDE);   // raw z
        const double *rc = reinterpret_cast<const double *>(smem + (j & 3) * RC::Q_STRIDE);         // raw z+1
        const double *sv = reinterpret_cast<const double *>(smem + RC::OFF_V + ((j - 1) & 1) * RC::V_STRIDE);
        double *rn = reinterpret_cast<double *>(smem + RC::OFF_N + (j & 1) * RC::N_STRIDE);         // q'(zc)
        unsigned pbo = LQ_BOND_PLAIN, pbh = LQ_BOND_PLAIN, pbo_prev = LQ_BOND_PLAIN;
        if (GEN) {
            // codes of plane zc sit in slot j & 3 (copied during iteration j-1), of plane zc-1 in slot (j-1) & 3;
            // a plane that is all plain was not copied: its codes are the constant
            if (ts[j - 2] == 0) {
                if (own_in) pbo = cown[(j & 3) * RC::NT];
                if (halo_in) pbh = chalo[(j & 3) * 128];
            }
            if (j >= 3 && ts[j - 3] == 0 && own_in) pbo_prev = cown[((j - 1) & 3) * RC::NT];
        }

        // ---- phase 1: F(q) and q' at (cx_, cy_) in q'-box coordinates; returns v_k for the own cell
        auto first = [&](int cx_, int cy_, unsigned code, double vk[5], double qn[5], bool own) {
            const int ridx = (cy_ + 1) * RC::RW + cx_ + 1;
            const int vidx = cy_ * RC::VW + cx_ + 1;
            const int gx = x0 - 1 + cx_, gy = y0 - 1 + cy_;
            double q5[5], F[5] = {0.0, 0.0, 0.0, 0.0, 0.0};
#pragma unroll
            for (int c = 0; c < 5; ++c) q5[c] = rb[c * RC::RPLANE + ridx];
            if (gx > a.g.Lx || gy > a.g.Ly) {       // ragged tile: beyond the ghost shell, never used
#pragma unroll
                for (int c = 0; c < 5; ++c) { vk[c] = 0.0; qn[c] = q5[c]; }
                return;
            }
            const bool sim = !GEN || !(code & LQ_BOND_OBJECT);
            if (sim) {
                double lap[5];
                if (!GEN || code == LQ_BOND_PLAIN) {
#pragma unroll
                    for (int c = 0; c < 5; ++c) {
                        const double *b = rb + c * RC::RPLANE + ridx;
                        lap[c] = ((b[-1] + b[1]) + (b[-RC::RW] + b[RC::RW]) +
                                  (ra[c * RC::RPLANE + ridx] + rc[c * RC::RPLANE + ridx])) - 6.0 * q5[c];
                    }
                } else {
                    const double w0 = lq_bond_weight(code, 0), w1 = lq_bond_weight(code, 1), w2 = lq_bond_weight(code, 2),
                                 w3 = lq_bond_weight(code, 3), w4 = lq_bond_weight(code, 4), w5 = lq_bond_weight(code, 5);
#pragma unroll
                    for (int c = 0; c < 5; ++c) {
                        const double *b = rb + c * RC::RPLANE + ridx;
                        const double qx = q5[c];
                        lap[c] = (w0 * (b[1] - qx) + w1 * (b[-1] - qx)) + (w2 * (b[RC::RW] - qx) + w3 * (b[-RC::RW] - qx)) +
                                 (w4 * (rc[c * RC::RPLANE + ridx] - qx) + w5 * (ra[c * RC::RPLANE + ridx] - qx));
                    }
                }
                lqs::bulk_force_oneconst(a.ph, q5, lap, F);
                if (GEN && (code & LQ_BOND_ANCH)) {
                    const F5 fa = anchor_force(a.ph, a.f, NP, a.g.pidx(gx, gy, zc), q5[0], q5[1], q5[2], q5[3], q5[4]);
                    F[0] += fa.a; F[1] += fa.b; F[2] += fa.c; F[3] += fa.d; F[4] += fa.e;
                }
            }
            if (FIRST && own && sim && active && zc >= zb && zc < ze) {
#pragma unroll
                for (int c = 0; c < 5; ++c) {
                    r0[0] = __fma_rn(F[c], F[c], r0[0]);
                    r0[1] = fmax(r0[1], fabs(F[c]));
                }
            }
#pragma unroll
            for (int c = 0; c < 5; ++c) {
                if (sim) drift(q5[c], sv[c * RC::VPLANE + vidx], F[c], ma, cF, dt, vk[c], qn[c]);
                else { vk[c] = 0.0; qn[c] = q5[c]; }
            }
        };
#pragma unroll
        for (int c = 0; c < 5; ++c) { qm[c] = qc[c]; qc[c] = qp[c]; vk0[c] = vk1[c]; }
        first(tx + 1, ty + 1, pbo, vk1, qp, true);
        {
            const int idx = (ty + 1) * RC::BXW + tx + 1;
#pragma unroll
            for (int c = 0; c < 5; ++c) rn[c * RC::PLANE + idx] = qp[c];
        }
        if (hx >= 0) {
            double vk[5], qn[5];
            first(hx, hy, pbh, vk, qn, false);
            const int idx = hy * RC::BXW + hx;
#pragma unroll
            for (int c = 0; c < 5; ++c) rn[c * RC::PLANE + idx] = qn[c];
        }
        // No barrier between the phases: phase 2 reads the q' slot written in the PREVIOUS iteration (ordered by
        // that iteration's closing barrier) and this thread's own registers, so both phases form one
        // instruction stream the scheduler can interleave.

        // ---- phase 2: F' = force(q'), second half kick, reductions, stores for plane k = zc - 1
        if (j >= 4 && active) {
            const int k = zc - 1;
            const double *rk = reinterpret_cast<const double *>(smem + RC::OFF_N + ((j - 1) & 1) * RC::N_STRIDE);
            const int idx = (ty + 1) * RC::BXW + tx + 1;
            const long long p = a.g.pidx(x, y, k);
            double Fn[5] = {0.0, 0.0, 0.0, 0.0, 0.0}, vn[5] = {0.0, 0.0, 0.0, 0.0, 0.0};
            const unsigned code = pbo_prev;
            const bool sim = !GEN || !(code & LQ_BOND_OBJECT);
            if (sim) {
                double lap[5];
                if (!GEN || code == LQ_BOND_PLAIN) {
#pragma unroll
                    for (int c = 0; c < 5; ++c) {
                        const double *b = rk + c * RC::PLANE + idx;
                        lap[c] = ((b[-1] + b[1]) + (b[-RC::BXW] + b[RC::BXW]) + (qm[c] + qp[c])) - 6.0 * qc[c];
                    }
                } else {
                    const double w0 = lq_bond_weight(code, 0), w1 = lq_bond_weight(code, 1), w2 = lq_bond_weight(code, 2),
                                 w3 = lq_bond_weight(code, 3), w4 = lq_bond_weight(code, 4), w5 = lq_bond_weight(code, 5);
#pragma unroll
                    for (int c = 0; c < 5; ++c) {
                        const double *b = rk + c * RC::PLANE + idx;
                        const double qx = qc[c];
                        lap[c] = (w0 * (b[1] - qx) + w1 * (b[-1] - qx)) + (w2 * (b[RC::BXW] - qx) + w3 * (b[-RC::BXW] - qx)) +
                                 (w4 * (qp[c] - qx) + w5 * (qm[c] - qx));
                    }
                }
                lqs::bulk_force_oneconst(a.ph, qc, lap, Fn);
                if (GEN && (code & LQ_BOND_ANCH)) {
                    const F5 fa = anchor_force(a.ph, a.f, NP, p, qc[0], qc[1], qc[2], qc[3], qc[4]);
                    Fn[0] += fa.a; Fn[1] += fa.b; Fn[2] += fa.c; Fn[3] += fa.d; Fn[4] += fa.e;
                }
#pragma unroll
                for (int c = 0; c < 5; ++c) {
                    vn[c] = __fma_rn(hdt, Fn[c], vk0[c]);
                    r[0] = __fma_rn(Fn[c], vn[c], r[0]);
                    r[1] = __fma_rn(Fn[c], Fn[c], r[1]);
                    r[2] = __fma_rn(vn[c], vn[c], r[2]);
                    r[3] = fmax(r[3], fabs(Fn[c]));
                }
            }
#pragma unroll
            for (int c = 0; c < 5; ++c) {
                a.qo[c * NP + p] = qc[c];
                a.vo[c * NP + p] = vn[c];
            }
            // periodic ghost shell of the outputs (width LQ_GH: the next sweep reads q with a 2-site halo)
            const int shx = ghost_shift(x, a.g.Lx, a.g.gwx), shy = ghost_shift(y, a.g.Ly, LQ_GH),
                      shz = ghost_shift_z(k, a.g);
            if (shx | shy | shz) {
                for (int m = 1; m < 8; ++m) {
                    if (((m & 1) && !shx) || ((m & 2) && !shy) || ((m & 4) && !shz)) continue;
                    const long long pg = p + ((m & 1) ? shx : 0) + ((m & 2) ? shy * a.g.sy : 0) + ((m & 4) ? shz * a.g.sz : 0);
#pragma unroll
                    for (int c = 0; c < 5; ++c) {
                        a.qo[c * NP + pg] = qc[c];
                        a.vo[c * NP + pg] = vn[c];
                    }
                }
            }
        }
    };

    for (int j = 0; j < nplanes; ++j) {
        if (MASKED) {
            // codes of plane zb+j-2 (phase 1 of the next iteration) -> slot (j+1) & 3
            if (j >= 1 && j + 1 < nplanes && ts[j - 1] == 0) {
                if (own_in) cp_async_4(cown + ((j + 1) & 3) * RC::NT, a.bond + a.g.pidx(x, y, zb + j - 2));
                if (halo_in) cp_async_4(chalo + ((j + 1) & 3) * 128, a.bond + a.g.pidx(x0 - 1 + hx, y0 - 1 + hy, zb + j - 2));
            }
            cp_async_commit();
        }
        mbar_wait(&full[j & 3], (j >> 2) & 1);
        if (j >= 2) {                              // the first stencil needs three raw planes
            if (MASKED && (ts[j - 2] == 0 || (j >= 3 && ts[j - 3] == 0))) {
                cp_async_wait_but_one();           // everything but this iteration's copy has landed
                body(std::true_type{}, j);
            } else {
                body(std::false_type{}, j);
            }
            // one barrier per plane: q' slot (j-1)&1 is rewritten by the next iteration's phase 1, and raw slot
            // (j-2)%4 / v slot (j-1)%2 are consumed by every thread: refill them with planes j+2
            __syncthreads();
            if (tid == 0 && j + 2 < nplanes) issue(j + 2);
        }
    }
    finish_step<RC::NT, FIRST>(a, sc, r, red, r0);
}

}  // namespace

int lq_sweep_rc_box(int which, int dim) {
    // TMA box dims: which 0 = q (36 x 20), 1 = vc (36 x 18)
    return dim == 0 ? RC::RW : (which == 0 ? RC::RH : RC::VH);
}
int lq_sweep_rc_tile(int dim) { return dim == 0 ? RC::TX : RC::TY; }
int lq_sweep_rc_max_chunk() { return RC::MAXZC; }

cudaError_t lq_launch_sweep_rc(bool masked, bool first, int ncta, bool *attr_set, const CUtensorMap &mq,
                               const CUtensorMap &mv, const lqsw::SweepArgs &a, cudaStream_t st) {
    const int variant = (masked ? 1 : 0) | (first ? 2 : 0);
    void (*kern)(const CUtensorMap, const CUtensorMap, const lqsw::SweepArgs) =
        variant == 0 ? k_sweep_rc<false, false> : variant == 1 ? k_sweep_rc<true, false>
      : variant == 2 ? k_sweep_rc<false, true> : k_sweep_rc<true, true>;
    if (!attr_set[variant]) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, RC::SMEM_BYTES);
        if (e != cudaSuccess) return e;
        attr_set[variant] = true;
    }
    kern<<<ncta, RC::NT, RC::SMEM_BYTES, st>>>(mq, mv, a);
    return cudaGetLastError();
}

// lq_sweep_rc.cu -- one-constant hot path with the force RECOMPUTED instead of stored (sm_100a).
//
// State carried between FIRE steps is only (q, vc): 4 x 5 fp64 per site-update = 160 B of compulsory
// HBM traffic; the force at q, needed for the lazy velocity rescale and the first half
// kick, is re-evaluated from q on the tile plus a one-site halo.  Per step and site
// (Algorithm 1):
//     F   = force(q)                               on tile + 1 halo   (needs q on tile + 2 halo)
//     v_k = mix_a vc + (mix_b + dt/2) F ; q' = q + dt v_k             on tile + 1 halo
//     F'  = force(q') ; vc' = v_k + dt/2 F' ; partial sums            on the tile
// Tiling: CTA = 32 x 16 columns marching over a z-chunk.  Per plane one elected thread issues two 4-D TMA
// boxes: q (36 x 20 x 1 x 5, start x0-2: the innermost start coordinate must be 16-byte aligned) into a
// 4-slot ring that doubles as the z-window of the first stencil, and vc (36 x 18 x 1 x 5) into a 2-slot
// stage; q' planes live in a 2-slot shared-memory ring and, for the thread's own column, in registers.
#include "lq_sweep.cuh"
#include "lq_sweep_dev.cuh"
#include "lq_site.cuh"

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
    static constexpr int OFF_TS = OFF_RED + 4 * (NT / 32) * 8;     // tile summaries of this CTA's planes (<= 80)
    static constexpr int SMEM_BYTES = OFF_TS + 128;
    static constexpr int NHALO = 2 * BXW + 2 * (BYH - 2);
};
static_assert(RC::SMEM_BYTES <= 232448, "shared memory budget");

template <bool MASKED>
__global__ void __launch_bounds__(RC::NT, 1)
k_sweep_rc(const __grid_constant__ CUtensorMap tq, const __grid_constant__ CUtensorMap tv, const SweepArgs a) {
    extern __shared__ __align__(1024) unsigned char smem[];
    const LqFireScalars sc = *a.sc;
    if (sc.converged) return;

    uint64_t *full = reinterpret_cast<uint64_t *>(smem + RC::OFF_BAR);   // [NQ]
    double *red = reinterpret_cast<double *>(smem + RC::OFF_RED);
    const int tid = threadIdx.x;
    const int tx = tid % RC::TX, ty = tid / RC::TX;
    const int x0 = blockIdx.x * RC::TX, y0 = blockIdx.y * RC::TY;
    const int zb = blockIdx.z * a.zc, ze = min(a.g.Lz, zb + a.zc);
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
        ts[tid] = a.tsum[((size_t)(zb + tid) * gridDim.y + blockIdx.y) * gridDim.x + blockIdx.x];
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

    // halo share: perimeter cell (hx, hy) of the 34 x 18 q' box; own cell is (tx+1, ty+1)
    int hx = -1, hy = -1;
    if (tid < RC::NHALO) {
        int h = tid;
        if (h < RC::BXW) { hx = h; hy = 0; }
        else if (h < 2 * RC::BXW) { hx = h - RC::BXW; hy = RC::BYH - 1; }
        else { h -= 2 * RC::BXW; hy = 1 + (h >> 1); hx = (h & 1) ? RC::BXW - 1 : 0; }
    }

    // per-site 'plain' bytes (1 plain, 0 non-plain simulated, 2 object) of the own cell and the halo cell,
    // fetched one iteration ahead so that no dependent global load gates a plane of a tile that touches
    // objects; phase 2 reuses the own-cell byte of the previous iteration (same plane)
    const bool own_in = x <= a.g.Lx && y <= a.g.Ly;
    const bool halo_in = hx >= 0 && x0 - 1 + hx <= a.g.Lx && y0 - 1 + hy <= a.g.Ly;
    unsigned pbo_next = 1u, pbh_next = 1u, pbo = 1u;
    for (int j = 0; j < nplanes; ++j) {
        const unsigned pbo_prev = pbo, pbh = pbh_next;
        pbo = pbo_next;
        pbo_next = pbh_next = 1u;
        if (MASKED && j >= 1 && j + 1 < nplanes && ts[j - 1] == 0) {
            if (own_in) pbo_next = a.plain[a.g.pidx(x, y, zb + j - 2)];
            if (halo_in) pbh_next = a.plain[a.g.pidx(x0 - 1 + hx, y0 - 1 + hy, zb + j - 2)];
        }
        mbar_wait(&full[j & 3], (j >> 2) & 1);
        if (j < 2) continue;                       // the first stencil needs three raw planes
        const int zc = zb + j - 3;                 // plane whose q' is produced now (zb-1 .. ze)
        const double *ra = reinterpret_cast<const double *>(smem + ((j - 2) & 3) * RC::Q_STRIDE);   // raw z-1
        const double *rb = reinterpret_cast<const double *>(smem + ((j - 1) & 3) * RC::Q_STRIDE);   // raw z
        const double *rc = reinterpret_cast<const double *>(smem + (j & 3) * RC::Q_STRIDE);         // raw z+1
        const double *sv = reinterpret_cast<const double *>(smem + RC::OFF_V + ((j - 1) & 1) * RC::V_STRIDE);
        double *rn = reinterpret_cast<double *>(smem + RC::OFF_N + (j & 1) * RC::N_STRIDE);         // q'(zc)

        // ---- phase 1: F(q) and q' at (cx_, cy_) in q'-box coordinates; returns v_k for the own cell
        auto first = [&](int cx_, int cy_, unsigned pb, double vk[5], double qn[5]) {
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
            const bool plain = !MASKED || pb == 1u, sim = !MASKED || pb != 2u;
            const long long p = (MASKED && !plain) ? a.g.pidx(gx, gy, zc) : 0;
            if (plain) {
                double lap[5];
#pragma unroll
                for (int c = 0; c < 5; ++c) {
                    const double *b = rb + c * RC::RPLANE + ridx;
                    lap[c] = ((b[-1] + b[1]) + (b[-RC::RW] + b[RC::RW]) +
                              (ra[c * RC::RPLANE + ridx] + rc[c * RC::RPLANE + ridx])) - 6.0 * q5[c];
                }
                lqs::bulk_force_oneconst(a.ph, q5, lap, F);
            } else if (sim) {
                // non-plain site: its force was computed by the fix-up kernel of the previous step
#pragma unroll
                for (int c = 0; c < 5; ++c) F[c] = a.Fi[c * NP + p];
            }
#pragma unroll
            for (int c = 0; c < 5; ++c) {
                if (sim) drift(q5[c], sv[c * RC::VPLANE + vidx], F[c], ma, cF, dt, vk[c], qn[c]);
                else { vk[c] = 0.0; qn[c] = q5[c]; }
            }
        };
#pragma unroll
        for (int c = 0; c < 5; ++c) { qm[c] = qc[c]; qc[c] = qp[c]; vk0[c] = vk1[c]; }
        first(tx + 1, ty + 1, pbo, vk1, qp);
        {
            const int idx = (ty + 1) * RC::BXW + tx + 1;
#pragma unroll
            for (int c = 0; c < 5; ++c) rn[c * RC::PLANE + idx] = qp[c];
        }
        if (hx >= 0) {
            double vk[5], qn[5];
            first(hx, hy, pbh, vk, qn);
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
            const bool plain = !MASKED || pbo_prev == 1u, sim = !MASKED || pbo_prev != 2u;
            if (sim) {
                if (plain) {
                    double lap[5];
#pragma unroll
                    for (int c = 0; c < 5; ++c) {
                        const double *b = rk + c * RC::PLANE + idx;
                        lap[c] = ((b[-1] + b[1]) + (b[-RC::BXW] + b[RC::BXW]) + (qm[c] + qp[c])) - 6.0 * qc[c];
                    }
                    lqs::bulk_force_oneconst(a.ph, qc, lap, Fn);
#pragma unroll
                    for (int c = 0; c < 5; ++c) {
                        vn[c] = __fma_rn(hdt, Fn[c], vk0[c]);
                        r[0] = __fma_rn(Fn[c], vn[c], r[0]);
                        r[1] = __fma_rn(Fn[c], Fn[c], r[1]);
                        r[2] = __fma_rn(vn[c], vn[c], r[2]);
                        r[3] = fmax(r[3], fabs(Fn[c]));
                    }
                } else {
                    // non-plain site: leave v_k in the velocity slot; the fix-up kernel adds dt/2 F'
#pragma unroll
                    for (int c = 0; c < 5; ++c) vn[c] = vk0[c];
                }
            }
#pragma unroll
            for (int c = 0; c < 5; ++c) {
                a.qo[c * NP + p] = qc[c];
                a.vo[c * NP + p] = vn[c];
            }
            // periodic ghost shell of the outputs (width LQ_GH: the next sweep reads q with a 2-site halo)
            const int shx = ghost_shift(x, a.g.Lx, LQ_GH), shy = ghost_shift(y, a.g.Ly, LQ_GH),
                      shz = ghost_shift(k, a.g.Lz, LQ_GH);
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
        // one barrier per plane: q' slot (j-1)&1 is rewritten by the next iteration's phase 1, and raw slot
        // (j-2)%4 / v slot (j-1)%2 are consumed by every thread: refill them with planes j+2
        __syncthreads();
        if (tid == 0 && j + 2 < nplanes) issue(j + 2);
    }
    finish_step<RC::NT>(a, sc, r, red);
}

}  // namespace

int lq_sweep_rc_box(int which, int dim) {
    // TMA box dims: which 0 = q (36 x 20), 1 = vc (36 x 18)
    return dim == 0 ? RC::RW : (which == 0 ? RC::RH : RC::VH);
}
int lq_sweep_rc_tile(int dim) { return dim == 0 ? RC::TX : RC::TY; }

cudaError_t lq_launch_sweep_rc(bool masked, dim3 grid, const CUtensorMap &mq, const CUtensorMap &mv,
                               const lqsw::SweepArgs &a, cudaStream_t st) {
    static bool attr[2] = {false, false};
    if (!attr[masked]) {
        cudaError_t e = masked ? cudaFuncSetAttribute(k_sweep_rc<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, RC::SMEM_BYTES)
                               : cudaFuncSetAttribute(k_sweep_rc<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, RC::SMEM_BYTES);
        if (e != cudaSuccess) return e;
        attr[masked] = true;
    }
    if (masked) k_sweep_rc<true><<<grid, RC::NT, RC::SMEM_BYTES, st>>>(mq, mv, a);
    else k_sweep_rc<false><<<grid, RC::NT, RC::SMEM_BYTES, st>>>(mq, mv, a);
    return cudaGetLastError();
}

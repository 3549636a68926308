// lq_resident.cu -- FIRE with the whole state resident ON CHIP (small one-constant lattices; sm_100a).
//
// The streaming sweeps (lq_sweep_rc.cu) are built for lattices that live in HBM; on a lattice of a few 10^4 sites
// (BASELINE.json config 1: 32^3 = 2.6 MB of state) one step of them is pure latency: a launch, a TMA pipeline fill
// per z-chunk, a tail.  Here ONE cooperative launch runs the whole lq_fire_minimize call: every CTA owns one brick of
// the lattice for the entire run, keeps q, v and the force of its sites in registers and the brick's q' (+ a one-site
// halo) in shared memory, and the only traffic per step is the brick surfaces through L2 and ONE grid barrier
// (Algorithm 1).  As in the streaming sweeps, q' of a site is a pointwise
// function of that site's (q, vc, F) and the step's global scalars, so a CTA recomputes the q' of its halo cells
// from its neighbours' state instead of waiting for them to publish it:
//     v_k = mix_a vc + (mix_b + dt/2) F ;  q' = q + dt v_k       own sites (registers) and halo cells (state of the
//                                                                 neighbour bricks, read from global buffer `in`)
//     F' = force(q') ;  vc' = v_k + dt/2 F'                      own sites; (q', vc', F') -> global buffer `out`
//     per-CTA (P, |F|^2, |v|^2, max|F|) -> global               block reduction in a fixed order
//     -- grid barrier --                                          (state and partials ping-pong by step parity)
//     every CTA reduces all CTAs' partials in index order and advances dt, alpha, N_pos (same bits everywhere)
// The stop test, the step cap and the initial-state test of Algorithm 1 are evaluated on the device; the host launches
// once and reads the scalars back.  Masked lattices: the per-site bond code (weighted 7-point stencil) and the
// anchoring record are loaded once and stay in registers.  Force and FIRE arithmetic are the same device functions
// the sweeps use (lqs::bulk_force_oneconst, lqs::anchoring, lqsw::drift, lq_fire_advance).
#include "lq_sweep.cuh"
#include "lq_sweep_dev.cuh"
#include "lq_site.cuh"
#include "../../include/lq.h"

#include <cooperative_groups.h>

namespace cg = cooperative_groups;

namespace {
using namespace lqsw;

struct ResArgs {
    LqGeom g;
    LqPhys ph;
    LqFields f;
    double *q[2], *v[2], *F[2];   // padded global state, ping-pong: step s reads buffer (cur + s) & 1, writes the other
    int cur;                // buffer that holds the initial q
    const uint32_t *bond;   // bond codes (masked lattices) or null
    LqFireScalars *sc;      // in: initial scalars; out: final scalars
    LqFireConsts fc;
    double *partials;       // [2][ncta][4] by step parity, then [ncta][2] for the initial state
    int nbx, nby, nbz;      // bricks per direction
    int bx, by, bz;         // brick size (the last brick of a direction may be ragged)
};

__device__ __forceinline__ int wrapi(int i, int L) { return i < 0 ? i + L : (i >= L ? i - L : i); }

template <int NT>
__global__ void __launch_bounds__(NT, 1) k_fire_resident(const ResArgs a) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cg::grid_group grid = cg::this_grid();
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    constexpr int NW = NT / 32;
    const int ncta = gridDim.x, cta = blockIdx.x;
    const int bxi = cta % a.nbx, byi = (cta / a.nbx) % a.nby, bzi = cta / (a.nbx * a.nby);
    const int x0 = bxi * a.bx, y0 = byi * a.by, z0 = bzi * a.bz;
    const int ex = min(a.bx, a.g.Lx - x0), ey = min(a.by, a.g.Ly - y0), ez = min(a.bz, a.g.Lz - z0);   // this brick's extent
    const int lx = tid % a.bx, ly = (tid / a.bx) % a.by, lz = tid / (a.bx * a.by);
    const bool active = lx < ex && ly < ey && lz < ez;
    const int SX = a.bx + 2, SY = a.by + 2, SZ = a.bz + 2, SP = SX * SY * SZ;      // shared box with halo
    double *qs = reinterpret_cast<double *>(smem_raw);                              // [5][SZ][SY][SX]
    double *red = qs + 5 * SP;                                                      // [4 * NW]
    __shared__ LqFireScalars s_sc;
    const long long NP = a.g.NP;
    const long long p = active ? a.g.pidx(x0 + lx, y0 + ly, z0 + lz) : 0;
    const int sidx = ((lz + 1) * SY + (ly + 1)) * SX + lx + 1;

    // per-site constants: bond code, anchoring record
    unsigned code = LQ_BOND_PLAIN;
    if (active && a.bond) code = a.bond[p];
    const bool sim = active && !(code & LQ_BOND_OBJECT);
    int akind = 0;
    double aW = 0.0, an[3] = {0.0, 0.0, 0.0};
    if (sim && (code & LQ_BOND_ANCH)) {
        akind = a.f.kind[p]; aW = a.f.W[p];
        an[0] = a.f.axis[p]; an[1] = a.f.axis[NP + p]; an[2] = a.f.axis[2 * NP + p];
    }
    const double w0 = lq_bond_weight(code, 0), w1 = lq_bond_weight(code, 1), w2 = lq_bond_weight(code, 2),
                 w3 = lq_bond_weight(code, 3), w4 = lq_bond_weight(code, 4), w5 = lq_bond_weight(code, 5);

    double q5[5], v5[5] = {0, 0, 0, 0, 0}, F5[5];
#pragma unroll
    for (int c = 0; c < 5; ++c) q5[c] = active ? a.q[a.cur][c * NP + p] : 0.0;

    // halo of the brick (the six faces; periodic index wrap): cell h -> global index pg and shared-box index si
    const int nf_xy = ex * ey, nf_xz = ex * ez, nf_yz = ey * ez, nhalo = 2 * (nf_xy + nf_xz + nf_yz);
    auto halo_cell = [&](int h, long long &pg, int &si) {
        int hx, hy, hz, t = h;
        if (t < 2 * nf_xy) { const int s = t >= nf_xy; t -= s * nf_xy; hx = t % ex; hy = t / ex; hz = s ? ez : -1; }
        else if ((t -= 2 * nf_xy) < 2 * nf_xz) { const int s = t >= nf_xz; t -= s * nf_xz; hx = t % ex; hz = t / ex; hy = s ? ey : -1; }
        else { t -= 2 * nf_xz; const int s = t >= nf_yz; t -= s * nf_yz; hy = t % ey; hz = t / ey; hx = s ? ex : -1; }
        pg = a.g.pidx(wrapi(x0 + hx, a.g.Lx), wrapi(y0 + hy, a.g.Ly), wrapi(z0 + hz, a.g.Lz));
        si = ((hz + 1) * SY + (hy + 1)) * SX + hx + 1;
    };
    // initial state: q of the halo cells as it stands (object cells keep this value for the whole run)
    auto load_halo = [&]() {
        for (int h = tid; h < nhalo; h += NT) {
            long long pg; int si;
            halo_cell(h, pg, si);
#pragma unroll
            for (int c = 0; c < 5; ++c) qs[c * SP + si] = __ldcg(a.q[a.cur] + c * NP + pg);
        }
    };
    // a step's q' of the halo cells, recomputed from the neighbours' (q, vc, F) in buffer `in` with the very
    // instruction sequence their owners use (lqsw::drift): no CTA waits for another one's q'.  The thread's first
    // halo cell (all of them when nhalo <= NT) is fetched into registers right after the grid barrier, so that its
    // L2 round trip overlaps the reduction of the partials.
    long long hp0 = -1; int hs0 = 0;                  // first halo cell: global index (-1: none or an object), box index
    if (tid < nhalo) {
        halo_cell(tid, hp0, hs0);
        if (a.bond && (a.bond[hp0] & LQ_BOND_OBJECT)) hp0 = -1;
    }
    double hq[5], hv[5], hF[5];
    auto fetch_halo0 = [&](int in) {
        if (hp0 < 0) return;
#pragma unroll
        for (int c = 0; c < 5; ++c) {
            hq[c] = __ldcg(a.q[in] + c * NP + hp0); hv[c] = __ldcg(a.v[in] + c * NP + hp0); hF[c] = __ldcg(a.F[in] + c * NP + hp0);
        }
    };
    auto drift_halo = [&](int in, const LqStepCoef &kc) {
        if (hp0 >= 0) {
#pragma unroll
            for (int c = 0; c < 5; ++c) {
                double vk, qn;
                drift(hq[c], hv[c], hF[c], kc.ma, kc.cF, kc.dt, vk, qn);
                qs[c * SP + hs0] = qn;
            }
        }
        for (int h = tid + NT; h < nhalo; h += NT) {
            long long pg; int si;
            halo_cell(h, pg, si);
            if (a.bond && (__ldg(a.bond + pg) & LQ_BOND_OBJECT)) continue;
#pragma unroll
            for (int c = 0; c < 5; ++c) {
                double vk, qn;
                drift(__ldcg(a.q[in] + c * NP + pg), __ldcg(a.v[in] + c * NP + pg), __ldcg(a.F[in] + c * NP + pg), kc.ma, kc.cF,
                      kc.dt, vk, qn);
                qs[c * SP + si] = qn;
            }
        }
    };
    // force on the own site from the shared box (weighted 7-point stencil + bulk + anchoring), same arithmetic as
    // the sweeps
    auto force = [&](const double qx[5], double F[5]) {
        double lap[5];
        if (code == LQ_BOND_PLAIN) {
#pragma unroll
            for (int c = 0; c < 5; ++c) {
                const double *b = qs + c * SP + sidx;
                lap[c] = ((b[-1] + b[1]) + (b[-SX] + b[SX]) + (b[-SX * SY] + b[SX * SY])) - 6.0 * qx[c];
            }
        } else {
#pragma unroll
            for (int c = 0; c < 5; ++c) {
                const double *b = qs + c * SP + sidx;
                const double qq = qx[c];
                lap[c] = (w0 * (b[1] - qq) + w1 * (b[-1] - qq)) + (w2 * (b[SX] - qq) + w3 * (b[-SX] - qq)) +
                         (w4 * (b[SX * SY] - qq) + w5 * (b[-SX * SY] - qq));
            }
        }
        lqs::bulk_force_oneconst(a.ph, qx, lap, F);
        if (akind != 0) {
            const double Q[6] = {qx[0], qx[1], qx[2], qx[3], qx[4], -qx[0] - qx[3]};
            double G[3][3] = {{0.0, 0.0, 0.0}, {0.0, 0.0, 0.0}, {0.0, 0.0, 0.0}};
            lqs::anchoring(a.ph, akind, aW, an, Q, G);
            double Fa[5];
            lqs::G_to_F(G, Fa);
#pragma unroll
            for (int c = 0; c < 5; ++c) F[c] += Fa[c];
        }
    };
    // block-reduce r (n entries; the first nsum are sums, the rest maxima) and publish at dst
    auto publish = [&](const double *r, int n, int nsum, double *dst) {
        for (int i = 0; i < n; ++i) {
            const double w = i < nsum ? warp_sum(r[i]) : warp_max(r[i]);
            if (lane == 0) red[i * NW + wid] = w;
        }
        __syncthreads();
        if (tid == 0)
            for (int i = 0; i < n; ++i) {
                double t = red[i * NW];
                for (int w = 1; w < NW; ++w) t = i < nsum ? t + red[i * NW + w] : fmax(t, red[i * NW + w]);
                dst[i] = t;
            }
        __syncthreads();
    };
    // every CTA: all CTAs' published values in index order -> tot (identical bits in every CTA)
    auto gather = [&](const double *src, int n, int nsum, double *tot) {
        double t[4] = {0.0, 0.0, 0.0, 0.0};
        for (int b = tid; b < ncta; b += NT)
            for (int i = 0; i < n; ++i) {
                const double x = __ldcg(src + n * b + i);
                t[i] = i < nsum ? t[i] + x : fmax(t[i], x);
            }
        for (int i = 0; i < n; ++i) {
            const double w = i < nsum ? warp_sum(t[i]) : warp_max(t[i]);
            if (lane == 0) red[i * NW + wid] = w;
        }
        __syncthreads();
        for (int i = 0; i < n; ++i) {
            double x = red[i * NW];
            for (int w = 1; w < NW; ++w) x = i < nsum ? x + red[i * NW + w] : fmax(x, red[i * NW + w]);
            tot[i] = x;
        }
        __syncthreads();
    };

    // ---- initial state: F(q_0) and Algorithm 1's stop test on it
    if (tid == 0) s_sc = *a.sc;
    if (active) {
#pragma unroll
        for (int c = 0; c < 5; ++c) qs[c * SP + sidx] = q5[c];
    }
    load_halo();
    __syncthreads();
#pragma unroll
    for (int c = 0; c < 5; ++c) F5[c] = 0.0;
    if (sim) force(q5, F5);
    if (active) {                                     // (vc = 0, F(q_0)) for the neighbours' first drift
#pragma unroll
        for (int c = 0; c < 5; ++c) { __stcg(a.v[a.cur] + c * NP + p, 0.0); __stcg(a.F[a.cur] + c * NP + p, F5[c]); }
    }
    {
        double r0[2] = {0.0, 0.0};
#pragma unroll
        for (int c = 0; c < 5; ++c) { r0[0] = __fma_rn(F5[c], F5[c], r0[0]); r0[1] = fmax(r0[1], fabs(F5[c])); }
        publish(r0, 2, 1, a.partials + 8 * ncta + 2 * cta);
        grid.sync();
        fetch_halo0(a.cur);
        double t0[4];
        gather(a.partials + 8 * ncta, 2, 1, t0);
        if (tid == 0) {
            LqFireScalars nx = s_sc;
            nx.P = 0.0; nx.FF = t0[0]; nx.vv = 0.0; nx.Fmax = t0[1];
            if (t0[1] < a.fc.force_tol) nx.converged = 1;
            s_sc = nx;
        }
        __syncthreads();
    }

    // ---- the FIRE loop, entirely on the device: one grid barrier per step
    int in = a.cur;
    while (!s_sc.converged && s_sc.step < a.fc.max_steps) {
        const LqFireScalars sc = s_sc;
        const LqStepCoef kc = lq_step_coef(sc, a.fc);
        const int out = in ^ 1;
        double vk[5], qn[5], Fn[5] = {0.0, 0.0, 0.0, 0.0, 0.0}, vn[5] = {0.0, 0.0, 0.0, 0.0, 0.0};
#pragma unroll
        for (int c = 0; c < 5; ++c) {
            if (sim) drift(q5[c], v5[c], F5[c], kc.ma, kc.cF, kc.dt, vk[c], qn[c]);
            else { vk[c] = 0.0; qn[c] = q5[c]; }
        }
        __syncthreads();                              // everyone is done reading the box of the previous step
        if (active) {
#pragma unroll
            for (int c = 0; c < 5; ++c) qs[c * SP + sidx] = qn[c];
        }
        drift_halo(in, kc);
        __syncthreads();
        double r[4] = {0.0, 0.0, 0.0, 0.0};
        if (sim) {
            force(qn, Fn);
#pragma unroll
            for (int c = 0; c < 5; ++c) {
                vn[c] = __fma_rn(kc.kick, Fn[c], vk[c]);
                r[0] = __fma_rn(Fn[c], vn[c], r[0]);
                r[1] = __fma_rn(Fn[c], Fn[c], r[1]);
                r[2] = __fma_rn(vn[c], vn[c], r[2]);
                r[3] = fmax(r[3], fabs(Fn[c]));
            }
        }
        if (active) {                                 // the new state, for the neighbours' next drift and the caller
#pragma unroll
            for (int c = 0; c < 5; ++c) {
                __stcg(a.q[out] + c * NP + p, qn[c]); __stcg(a.v[out] + c * NP + p, vn[c]); __stcg(a.F[out] + c * NP + p, Fn[c]);
            }
        }
        double *part = a.partials + (size_t)out * 4 * ncta;   // by parity: a fast CTA may publish step s+1 while a slow one gathers s
        publish(r, 4, 3, part + 4 * cta);
        grid.sync();
        fetch_halo0(out);
        double tot[4];
        gather(part, 4, 3, tot);
        if (tid == 0) {
            LqFireScalars nx = sc;
            lq_fire_advance(nx, a.fc, tot, 0);
            s_sc = nx;
        }
#pragma unroll
        for (int c = 0; c < 5; ++c) { q5[c] = qn[c]; v5[c] = vn[c]; F5[c] = Fn[c]; }
        in = out;
        __syncthreads();
    }

    // ---- results: q, vc of the final state sit in buffer (cur + steps) & 1; scalars
    if (cta == 0 && tid == 0) *a.sc = s_sc;
}

}  // namespace

// Can this lattice run resident, and with what bricks?  Picks brick counts (nbx, nby, nbz) with nbx*nby*nbz <= nsm
// and brick volume <= 512 sites that minimise the thread count per CTA (most parallelism), then the number of bricks,
// then the brick surface.
bool lq_resident_plan(const LqGeom &g, int nsm, int dims[6]) {
    long long best_vol = -1, best_surf = 0, best_n = 0;
    for (int nbz = 1; nbz <= g.Lz; ++nbz)
        for (int nby = 1; nby <= g.Ly && (long long)nbz * nby <= nsm; ++nby)
            for (int nbx = 1; nbx <= g.Lx && (long long)nbz * nby * nbx <= nsm; ++nbx) {
                const int bx = (g.Lx + nbx - 1) / nbx, by = (g.Ly + nby - 1) / nby, bz = (g.Lz + nbz - 1) / nbz;
                // no empty bricks; a periodic halo needs at least 2 bricks or the whole axis, and bricks >= 2 wide
                if ((long long)bx * (nbx - 1) >= g.Lx || (long long)by * (nby - 1) >= g.Ly || (long long)bz * (nbz - 1) >= g.Lz) continue;
                const long long vol = (long long)bx * by * bz;
                if (vol > 512) continue;
                const long long volr = ((vol + 127) / 128) * 128;                   // thread-count granularity
                const long long surf = 2LL * (bx * by + bx * bz + by * bz);
                const long long n = (long long)nbx * nby * nbz;
                if (best_vol < 0 || volr < best_vol || (volr == best_vol && (n < best_n || (n == best_n && surf < best_surf)))) {
                    best_vol = volr; best_surf = surf; best_n = n;
                    dims[0] = nbx; dims[1] = nby; dims[2] = nbz; dims[3] = bx; dims[4] = by; dims[5] = bz;
                }
            }
    return best_vol > 0;
}

// One cooperative launch = the whole minimisation.  Returns cudaErrorCooperativeLaunchTooLarge (or another error) if
// the grid cannot be co-resident; the caller then falls back to the streaming sweeps.
cudaError_t lq_launch_fire_resident(const LqGeom &g, const LqPhys &ph, const LqFields &f, double *const q[2],
                                    double *const v[2], double *const F[2], int cur, const uint32_t *bond,
                                    LqFireScalars *sc, const LqFireConsts &fc, double *partials, const int dims[6],
                                    cudaStream_t st) {
    ResArgs a;
    a.g = g; a.ph = ph; a.f = f; a.bond = bond; a.sc = sc; a.fc = fc; a.partials = partials; a.cur = cur;
    for (int i = 0; i < 2; ++i) { a.q[i] = q[i]; a.v[i] = v[i]; a.F[i] = F[i]; }
    a.nbx = dims[0]; a.nby = dims[1]; a.nbz = dims[2]; a.bx = dims[3]; a.by = dims[4]; a.bz = dims[5];
    const int vol = a.bx * a.by * a.bz;
    const int nt = vol <= 128 ? 128 : (vol <= 256 ? 256 : 512);
    const int ncta = a.nbx * a.nby * a.nbz;
    const size_t smem = (size_t)5 * (a.bx + 2) * (a.by + 2) * (a.bz + 2) * sizeof(double) + (size_t)4 * (nt / 32) * sizeof(double);
    void *kern = nt == 128 ? (void *)k_fire_resident<128> : (nt == 256 ? (void *)k_fire_resident<256> : (void *)k_fire_resident<512>);
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    int per_sm = 0, dev = 0, nsm = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev);
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, nt, smem);
    if (e != cudaSuccess) return e;
    if ((long long)per_sm * nsm < ncta) return cudaErrorCooperativeLaunchTooLarge;
    void *args[] = {(void *)&a};
    return cudaLaunchCooperativeKernel(kern, dim3(ncta), dim3(nt), args, smem, st);
}

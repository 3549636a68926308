// lq_sweep.cu -- the hot path: ONE kernel launch per FIRE step (sm_100a).
//
// State carried between steps is (q, vc, F): the Q field, the velocity after the second
// half-kick (before the rescale), and the force at q.  Step n+1, per site
// (Algorithm 1):
//     v_m = mix_a vc + mix_b F                    velocity rescale decided by step n's reductions
//     v_k = v_m + dt/2 F ;  q' = q + dt v_k       half kick + drift
//     F'  = force(q')                             bulk + elastic stencil + anchoring (fused)
//     vc' = v_k + dt/2 F'                         second half kick
//     partial sums of F'.vc', |F'|^2, |vc'|^2, max|F'_a|
// q' of a site is a pointwise function of that site's (q, vc, F) and three global scalars, so a CTA
// recomputes q' on its tile PLUS a one-site halo from TMA-staged boxes of the three input fields and
// never needs a neighbour CTA's output: no second pass, no grid barrier.  The last CTA to finish
// reduces the per-CTA partials in a fixed order and advances the FIRE schedule on the device.
//
// Tiling: CTA = TX x TY columns marching over a z-chunk.  Per plane, one elected thread issues three
// 4-D TMA box loads ((TX+4) x (TY+2) x 1 x 5 components) into a 2-stage mbarrier ring; all threads turn
// the landed plane into q' (own site + a share of the halo ring) in a 3-plane shared-memory ring; the
// force for plane k then reads its in-plane neighbours from shared memory and its z neighbours from
// registers.  Outputs go straight from registers to global memory with coalesced 256-byte rows; sites
// on the lattice faces also refresh the periodic ghost shell of the output buffers.
#include "lq_sweep.cuh"
#include "lq_sweep_dev.cuh"
#include "lq_site.cuh"
#include "../../include/lq.h"

#include <cuda.h>
#include <cstdio>
#include <cstring>
#include <algorithm>
#include <functional>
#include <queue>
#include <vector>

namespace {
using namespace lqsw;

template <int TX_, int TY_>
struct Cfg {
    static constexpr int TX = TX_, TY = TY_, NT = TX_ * TY_;
    static constexpr int BXW = TX_ + 2, BYH = TY_ + 2;      // q' ring: tile + 1 halo
    static constexpr int PLANE = BXW * BYH;                 // elements of one component plane of the ring
    static constexpr int RING_STRIDE = (5 * PLANE * 8 + 127) / 128 * 128;
    // TMA box: the start coordinate of the innermost dimension must be 16-byte aligned (measured: an odd
    // fp64 start coordinate traps with "illegal instruction"), so the staged box starts at x0-2, not x0-1.
    static constexpr int SW = TX_ + 4;                      // staged box width: x0-2 .. x0+TX+1
    static constexpr int SPLANE = SW * BYH;
    static constexpr int FIELD_BYTES = 5 * SPLANE * 8;      // one TMA box
    static constexpr int FIELD_STRIDE = (FIELD_BYTES + 127) / 128 * 128;
    static constexpr int NSTAGE = 2, RING = 3;
    static constexpr int STAGE_BYTES = 3 * FIELD_STRIDE;
    static constexpr int OFF_RING = NSTAGE * STAGE_BYTES;
    static constexpr int OFF_BAR = OFF_RING + RING * RING_STRIDE;
    static constexpr int OFF_RED = OFF_BAR + 64;
    static constexpr int OFF_TS = OFF_RED + 4 * (NT / 32) * 8;     // tile summaries of this CTA's planes
    static constexpr int SMEM_BYTES = OFF_TS + 128;
    static constexpr int NHALO = 2 * BXW + 2 * (BYH - 2);
};

// XT: extra distortion terms compiled into the 19-point stencil (bit 0 chiral L4, bit 1 cubic L6)
template <class C, bool THREE, bool MASKED, int XT>
__global__ void __launch_bounds__(C::NT, 1)
k_sweep(const __grid_constant__ CUtensorMap tq, const __grid_constant__ CUtensorMap tv,
        const __grid_constant__ CUtensorMap tF, const SweepArgs a) {
    extern __shared__ __align__(1024) unsigned char smem[];
    constexpr bool TWO_SYNC = THREE || MASKED;   // the general force reads ring plane k-1 too
    const LqFireScalars sc = *a.sc;
    if (sc.converged) return;

    uint64_t *full = reinterpret_cast<uint64_t *>(smem + C::OFF_BAR);
    double *red = reinterpret_cast<double *>(smem + C::OFF_RED);
    const int tid = threadIdx.x;
    const int tx = tid % C::TX, ty = tid / C::TX;
    const int4 wk = a.work[blockIdx.x];          // (tile x, tile y, first plane, end plane), longest items first
    const int x0 = wk.x * C::TX, y0 = wk.y * C::TY;
    const int zb = wk.z, ze = wk.w;
    const int x = x0 + tx, y = y0 + ty;
    const bool active = x < a.g.Lx && y < a.g.Ly;
    const int nplanes = ze - zb + 2;             // planes zb-1 .. ze
    const long long NP = a.g.NP;

    if (tid == 0) {
        mbar_init(&full[0], 1);
        mbar_init(&full[1], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    uint8_t *ts = smem + C::OFF_TS;               // ts[i] = summary of plane zb+i
    if (MASKED && tid < ze - zb)
        ts[tid] = a.tsum[((size_t)(zb + tid + 1) * a.nty + wk.y) * a.ntx + wk.x];
    __syncthreads();

    auto issue = [&](int j) {
        const int s = j & 1;
        unsigned char *st = smem + s * C::STAGE_BYTES;
        const int cx = x0 + LQ_XO - 2, cy = y0 + LQ_GH - 1, cz = zb - 1 + j + LQ_GH;
        mbar_expect_tx(&full[s], 3u * C::FIELD_BYTES);
        tma_load_4d(st, &tq, &full[s], cx, cy, cz, 0);
        tma_load_4d(st + C::FIELD_STRIDE, &tv, &full[s], cx, cy, cz, 0);
        tma_load_4d(st + 2 * C::FIELD_STRIDE, &tF, &full[s], cx, cy, cz, 0);
    };
    if (tid == 0) {
        issue(0);
        if (nplanes > 1) issue(1);
    }

    const LqStepCoef kc = lq_step_coef(sc, a.fc);
    const double dt = kc.dt, ma = kc.ma, cF = kc.cF, hdt = kc.kick;
    double qm[5], qc[5], qp[5], vk0[5], vk1[5];
#pragma unroll
    for (int c = 0; c < 5; ++c) qm[c] = qc[c] = qp[c] = vk0[c] = vk1[c] = 0.0;
    double r[4] = {0.0, 0.0, 0.0, 0.0};
    const int idx = (ty + 1) * C::BXW + tx + 1;    // own site in a ring plane
    const int sidx = (ty + 1) * C::SW + tx + 2;    // own site in a staged box

    // halo share of this thread: perimeter cell h of the (TX+2) x (TY+2) box
    int hidx = -1, hsidx = -1;
    if (tid < C::NHALO) {
        int h = tid, hx, hy;
        if (h < C::BXW) { hx = h; hy = 0; }
        else if (h < 2 * C::BXW) { hx = h - C::BXW; hy = C::BYH - 1; }
        else { h -= 2 * C::BXW; hy = 1 + (h >> 1); hx = (h & 1) ? C::BXW - 1 : 0; }
        hidx = hy * C::BXW + hx;
        hsidx = hy * C::SW + hx + 1;
    }

    // per-site 'plain' byte of the plane phase B handles, fetched one iteration ahead (1 plain, 0 non-plain
    // simulated, 2 object): no dependent global load sits on the critical path of tiles that touch objects
    unsigned pb_next = 1u;
    for (int j = 0; j < nplanes; ++j) {
        const int s = j & 1;
        const unsigned pb = pb_next;
        pb_next = 1u;
        if (MASKED && active && j >= 1 && j + 1 < nplanes && ts[j - 1] == 0) pb_next = a.plain[a.g.pidx(x, y, zb + j - 1)];
        mbar_wait(&full[s], (j >> 1) & 1);
        const double *sq = reinterpret_cast<const double *>(smem + s * C::STAGE_BYTES);
        const double *sv = sq + C::FIELD_STRIDE / 8, *sF = sq + 2 * (C::FIELD_STRIDE / 8);
        double *rn = reinterpret_cast<double *>(smem + C::OFF_RING + (j % 3) * C::RING_STRIDE);

        // ---- [A] plane z = zb-1+j: q' on tile + halo into the ring; own column into registers
#pragma unroll
        for (int c = 0; c < 5; ++c) {
            qm[c] = qc[c]; qc[c] = qp[c]; vk0[c] = vk1[c];
            drift(sq[c * C::SPLANE + sidx], sv[c * C::SPLANE + sidx], sF[c * C::SPLANE + sidx], ma, cF, dt, vk1[c], qp[c]);
            rn[c * C::PLANE + idx] = qp[c];
        }
        if (hidx >= 0) {
#pragma unroll
            for (int c = 0; c < 5; ++c) {
                double vk, qn;
                drift(sq[c * C::SPLANE + hsidx], sv[c * C::SPLANE + hsidx], sF[c * C::SPLANE + hsidx], ma, cF, dt, vk, qn);
                rn[c * C::PLANE + hidx] = qn;
            }
        }
        __syncthreads();
        if (tid == 0 && j + 2 < nplanes) issue(j + 2);   // stage s has been consumed by every thread

        // ---- [B] force, second half kick, reductions and stores for plane k = zb + j - 2
        if (j >= 2 && active) {
            const int k = zb + j - 2;
            const bool tile_plain = !MASKED || ts[k - zb] != 0;
            const double *rk = reinterpret_cast<const double *>(smem + C::OFF_RING + ((j - 1) % 3) * C::RING_STRIDE);
            const long long p = a.g.pidx(x, y, k);
            double Fn[5] = {0.0, 0.0, 0.0, 0.0, 0.0}, vn[5] = {0.0, 0.0, 0.0, 0.0, 0.0};
            // plain: constant stencil weights
            const bool plain = !MASKED || tile_plain || pb == 1u;
            const bool sim = !MASKED || tile_plain || pb != 2u;
            if (sim) {
                if (plain) {
                    if (!THREE) {
                        double lap[5];
#pragma unroll
                        for (int c = 0; c < 5; ++c) {
                            const double *b = rk + c * C::PLANE + idx;
                            lap[c] = ((b[-1] + b[1]) + (b[-C::BXW] + b[C::BXW]) + (qm[c] + qp[c])) - 6.0 * qc[c];
                        }
                        lqs::bulk_force_oneconst(a.ph, qc, lap, Fn);
                    } else {
                        const double *rkm = reinterpret_cast<const double *>(smem + C::OFF_RING + ((j - 2) % 3) * C::RING_STRIDE);
                        auto get = [&](int c, int dx, int dy, int dz) -> double {
                            if (dz == 0) return rk[c * C::PLANE + idx + dy * C::BXW + dx];
                            if (dx == 0 && dy == 0) return dz < 0 ? qm[c] : qp[c];
                            return (dz < 0 ? rkm : rn)[c * C::PLANE + idx + dy * C::BXW + dx];
                        };
                        lqs::bulk_force_threeconst<(XT & 1) != 0, (XT & 2) != 0>(a.ph, get, qc, Fn);
                    }
#pragma unroll
                    for (int c = 0; c < 5; ++c) {
                        vn[c] = __fma_rn(hdt, Fn[c], vk0[c]);
                        r[0] = __fma_rn(Fn[c], vn[c], r[0]);
                        r[1] = __fma_rn(Fn[c], Fn[c], r[1]);
                        r[2] = __fma_rn(vn[c], vn[c], r[2]);
                        r[3] = fmax(r[3], fabs(Fn[c]));
                    }
                } else {
                    // non-plain site: leave v_k in the velocity slot; the fix-up kernel computes F', adds
                    // dt/2 F' and writes the force slot (and both ghost images)
#pragma unroll
                    for (int c = 0; c < 5; ++c) vn[c] = vk0[c];
                }
            }
            const bool store_F = !(sim && !plain);
#pragma unroll
            for (int c = 0; c < 5; ++c) {
                a.qo[c * NP + p] = qc[c];
                a.vo[c * NP + p] = vn[c];
                if (store_F) a.Fo[c * NP + p] = Fn[c];
            }
            // periodic ghost shell of the outputs, full width LQ_GH: whatever runs next on this state (the
            // recompute sweep reads q with a 2-site halo) finds every ghost current
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
                        if (store_F) a.Fo[c * NP + pg] = Fn[c];
                    }
                }
            }
        }
        if (TWO_SYNC) __syncthreads();
    }

    lqsw::finish_step<C::NT>(a, sc, r, red);
}

// ---------------------------------------------------------------- host side
typedef CUresult (*PFN_encodeTiled)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                    const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                    CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

PFN_encodeTiled get_encode() {
    static PFN_encodeTiled fn = nullptr;
    if (fn) return fn;
    void *p = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) != cudaSuccess ||
        q != cudaDriverEntryPointSuccess)
        return nullptr;
    fn = (PFN_encodeTiled)p;
    return fn;
}

bool make_map(CUtensorMap *m, const LqGeom &g, double *base, int bxw, int byh) {
    PFN_encodeTiled enc = get_encode();
    if (!enc) return false;
    cuuint64_t dims[4] = {(cuuint64_t)g.Px, (cuuint64_t)g.Py, (cuuint64_t)g.Pz, 5};
    cuuint64_t strides[3] = {(cuuint64_t)g.Px * 8, (cuuint64_t)g.sz * 8, (cuuint64_t)g.NP * 8};
    cuuint32_t box[4] = {(cuuint32_t)bxw, (cuuint32_t)byh, 1, 5};
    cuuint32_t es[4] = {1, 1, 1, 1};
    return enc(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 4, base, dims, strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
               CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) ==
           CUDA_SUCCESS;
}

}  // namespace

bool lq_make_box_map(CUtensorMap *m, const LqGeom &g, double *base, int bxw, int byh) { return make_map(m, g, base, bxw, byh); }

struct LqSweepPlan {
    CUtensorMap mq[2], mv[2], mF[2];
    double *bq[2] = {nullptr, nullptr}, *bv[2] = {nullptr, nullptr}, *bF[2] = {nullptr, nullptr};
    bool three = false, stored = true;
    double *partials = nullptr, *partials0 = nullptr;
    unsigned int *counter = nullptr;
    uint8_t *plain = nullptr, *tsum = nullptr;   // masked lattices: per-site and per-(plane, tile) 'plain' maps
    uint32_t *bond = nullptr;                    // recompute path on masked lattices: per-site bond codes
    int *np_list = nullptr;                      // stored path: index-ordered non-plain simulated sites (fix-up kernel)
    int n_np = 0;
    double *partials2 = nullptr;
    unsigned int *counter2 = nullptr;
    const uint8_t *flags_seen = nullptr, *kind_seen = nullptr;
    bool sites_dirty = true;
    int4 *work = nullptr;                        // work items (tile, z-range), longest first
    int n_items = 0, ntx = 0, nty = 0, chunks_forced = 0, ty = 0;
    bool attr_set[12] = {}, attr_rc[4] = {};
};

void lq_sweep_destroy(LqSweepPlan *p) {
    if (!p) return;
    cudaFree(p->partials);
    cudaFree(p->partials0);
    cudaFree(p->counter);
    cudaFree(p->plain);
    cudaFree(p->tsum);
    cudaFree(p->bond);
    cudaFree(p->np_list);
    cudaFree(p->partials2);
    cudaFree(p->counter2);
    cudaFree(p->work);
    delete p;
}
void lq_sweep_invalidate(LqSweepPlan *p) {
    if (p) p->sites_dirty = true;
}

// Work table of the recompute sweep: every tile column (ntiles of them, Lz planes each) is cut into z-chunks; a
// CTA pays its chunk plus `ovh` planes of halo and pipeline fill, one CTA per SM.  With few tiles per SM, equal
// chunks waste most of the last wave (config 5: 650 equal CTAs on 148 SMs = 4.4 waves of work in 5), so the first
// Ta tiles get na chunks and the rest nb >= na chunks, items are ordered longest first -- the hardware hands CTA
// ids out in order as SMs free up, i.e. longest-processing-time list scheduling -- and (Ta, na, nb) minimise the
// simulated makespan.  Large grids (many waves) keep equal chunks of <= 64 planes.
std::vector<int4> lq_build_chunk_table(int ntx, int nty, int Lz, int max_chunk, int ovh, int nsm, int force_n) {
    const int T = ntx * nty;
    auto chunks = [&](int n, int i, int &zb, int &ze) {      // i-th of n near-equal chunks of [0, Lz)
        zb = (int)((long long)Lz * i / n); ze = (int)((long long)Lz * (i + 1) / n);
    };
    const int n_min = (Lz + max_chunk - 1) / max_chunk;      // fewest chunks per column
    const int n_max = Lz >= 8 ? Lz / 4 : 1;                   // chunks of at least 4 planes
    int best_na = (Lz + 63) / 64, best_nb = best_na, best_Ta = T;
    if (best_na > n_max) best_na = best_nb = n_max;
    if (best_na < n_min) best_na = best_nb = n_min;
    if (force_n > 0) {                                        // "rc_chunks" option: n equal chunks per column
        best_na = best_nb = std::min(std::max(force_n, n_min), std::max(n_max, n_min));
    } else if ((long long)T * best_na < 10LL * nsm) {
        double best = -1.0;
        std::vector<long long> load(nsm);
        // a candidate's cost multiset depends only on the chunk lengths: histogram them (no sort), and skip the
        // candidate when its lower bound max(ceil(sum / nsm), longest item) cannot beat the best makespan so far
        // (only a strictly smaller makespan replaces the best, so the table chosen is the same as an exhaustive
        // search's).  This is host time of the first call on a context.
        std::vector<int> hist((size_t)Lz + ovh + 2);
        auto add_lengths = [&](int n, long long tiles, int &longest) {
            if (tiles <= 0) return;
            for (int i = 0; i < n; ++i) {
                int zb, ze;
                chunks(n, i, zb, ze);
                hist[ze - zb + ovh] += (int)tiles;
                if (ze - zb + ovh > longest) longest = ze - zb + ovh;
            }
        };
        auto makespan = [&](int Ta, int na, int nb) -> double {
            // items: Ta*na of cost ~Lz/na + ovh, (T-Ta)*nb of cost ~Lz/nb + ovh; longest first, each onto the
            // least-loaded SM
            const long long sum = (long long)Ta * (Lz + (long long)na * ovh) + (long long)(T - Ta) * (Lz + (long long)nb * ovh);
            std::fill(hist.begin(), hist.end(), 0);
            int longest = 0;
            add_lengths(na, Ta, longest);
            add_lengths(nb, T - Ta, longest);
            const long long lb = std::max((sum + nsm - 1) / nsm, (long long)longest);
            if (best >= 0.0 && (double)lb >= best) return (double)lb;      // cannot be strictly better
            std::priority_queue<long long, std::vector<long long>, std::greater<long long>> pq(std::greater<long long>(), load);
            long long mk = 0;
            for (int c = longest; c >= 0; --c)
                for (int k = 0; k < hist[c]; ++k) { long long l = pq.top() + c; pq.pop(); pq.push(l); if (l > mk) mk = l; }
            return (double)mk;
        };
        for (int na = n_min; na <= n_max && na <= n_min + 24; ++na)
            for (int nb = na; nb <= n_max && nb <= 4 * na + 4; ++nb) {
                for (int Ta = 0; Ta <= T; Ta += (Ta + nsm <= T ? nsm : (Ta < T ? T - Ta : 1))) {
                    if (nb == na && Ta != T) continue;
                    if ((long long)Ta * na + (long long)(T - Ta) * nb > 40LL * nsm) continue;
                    const double m = makespan(Ta, na, nb);
                    if (best < 0.0 || m < best) { best = m; best_na = na; best_nb = nb; best_Ta = Ta; }
                }
            }
    }
    std::vector<int4> items;
    for (int t = 0; t < T; ++t) {
        const int n = t < best_Ta ? best_na : best_nb;
        for (int i = 0; i < n; ++i) {
            int zb, ze;
            chunks(n, i, zb, ze);
            if (ze > zb) items.push_back(make_int4(t % ntx, t / ntx, zb, ze));
        }
    }
    // longest first; equal lengths: by z-chunk, then row-major tiles (x-neighbours share halo rows in L2)
    std::stable_sort(items.begin(), items.end(), [](const int4 &a, const int4 &b) {
        const int la = a.w - a.z, lb = b.w - b.z;
        if (la != lb) return la > lb;
        if (a.z != b.z) return a.z < b.z;
        if (a.y != b.y) return a.y < b.y;
        return a.x < b.x;
    });
    return items;
}

template <class C, bool THREE, bool MASKED, int XT = 0>
static cudaError_t launch(LqSweepPlan *pl, int in, const SweepArgs &a, int variant, cudaStream_t st) {
    if (!pl->attr_set[variant]) {
        cudaError_t e = cudaFuncSetAttribute(k_sweep<C, THREE, MASKED, XT>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                             C::SMEM_BYTES);
        if (e != cudaSuccess) return e;
        pl->attr_set[variant] = true;
    }
    k_sweep<C, THREE, MASKED, XT><<<pl->n_items, C::NT, C::SMEM_BYTES, st>>>(pl->mq[in], pl->mv[in], pl->mF[in], a);
    return cudaGetLastError();
}

#define LQ_PLAN_CUDA(call)                                                                   \
    do {                                                                                     \
        cudaError_t e_ = (call);                                                             \
        if (e_ != cudaSuccess) {                                                             \
            err = std::string("lq_sweep: " #call ": ") + cudaGetErrorString(e_);             \
            return e_ == cudaErrorMemoryAllocation ? LQ_ERR_NOMEM : LQ_ERR_CUDA;             \
        }                                                                                    \
    } while (0)

int lq_sweep_prepare(LqSweepPlan **planp, bool stored_F, const LqGeom &g, const LqPhys &ph, const LqFields &f, double *q[2],
                     double *v[2], double *F[2], cudaStream_t st, long *launches, std::string &err, int rc_chunks) {
    const bool three = lq_three(ph);
    const bool masked = f.flags != nullptr;
    LqSweepPlan *pl = *planp;
    if (!pl) {
        pl = new LqSweepPlan();
        *planp = pl;
    }
    if (three && !stored_F) { err = "lq_sweep: the recompute path is one-constant only"; return LQ_ERR_ARG; }
    // stored-force sweep: 32 x 16 tiles; with the cubic term (L6) 32 x 8 tiles of 256 threads, whose 255-register
    // budget holds the 19-point cubic stencil without spills
    const int TX = 32, TY = !stored_F ? lq_sweep_rc_tile(1) : (ph.L6 != 0.0 ? 8 : 16);
    bool rebuild = pl->three != three || pl->stored != stored_F || pl->partials == nullptr || pl->chunks_forced != rc_chunks ||
                   pl->ty != TY;
    pl->chunks_forced = rc_chunks;
    pl->ty = TY;
    for (int i = 0; i < 2; ++i) rebuild |= pl->bq[i] != q[i] || pl->bv[i] != v[i] || (stored_F && pl->bF[i] != F[i]);
    if (rebuild) {
        for (int i = 0; i < 2; ++i) {
            const bool ok = stored_F
                ? make_map(&pl->mq[i], g, q[i], TX + 4, TY + 2) && make_map(&pl->mv[i], g, v[i], TX + 4, TY + 2) &&
                  make_map(&pl->mF[i], g, F[i], TX + 4, TY + 2)
                : make_map(&pl->mq[i], g, q[i], lq_sweep_rc_box(0, 0), lq_sweep_rc_box(0, 1)) &&
                  make_map(&pl->mv[i], g, v[i], lq_sweep_rc_box(1, 0), lq_sweep_rc_box(1, 1));
            if (!ok) {
                err = "lq_sweep: cuTensorMapEncodeTiled failed";
                return LQ_ERR_CUDA;
            }
            pl->bq[i] = q[i]; pl->bv[i] = v[i]; pl->bF[i] = F[i];
        }
        pl->three = three;
        pl->stored = stored_F;
        const int ntx = (g.Lx + TX - 1) / TX, nty = (g.Ly + TY - 1) / TY;
        pl->ntx = ntx; pl->nty = nty;
        // z-chunks per tile column: the work table of lq_build_chunk_table (both sweeps; a chunk costs its planes
        // plus the halo planes and the pipeline fill: 4 + 3 for the recompute sweep, 2 + 3 for the stored-force one,
        // whose tile-summary array caps a chunk at 128 planes)
        int nsm = 148;
        int dev = 0;
        if (cudaGetDevice(&dev) == cudaSuccess) cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev);
        const std::vector<int4> items = stored_F ? lq_build_chunk_table(ntx, nty, g.Lz, 126, 5, nsm, rc_chunks)
                                                 : lq_build_chunk_table(ntx, nty, g.Lz, lq_sweep_rc_max_chunk(), 7, nsm, rc_chunks);
        cudaFree(pl->work); pl->work = nullptr;
        LQ_PLAN_CUDA(cudaMalloc(&pl->work, items.size() * sizeof(int4)));
        // pageable host source: the copy is staged before the call returns, `items` may go out of scope
        LQ_PLAN_CUDA(cudaMemcpyAsync(pl->work, items.data(), items.size() * sizeof(int4), cudaMemcpyHostToDevice, st));
        pl->n_items = (int)items.size();
        const size_t ncta = items.size();
        cudaFree(pl->partials); cudaFree(pl->partials0); cudaFree(pl->counter);
        pl->partials = pl->partials0 = nullptr; pl->counter = nullptr;
        LQ_PLAN_CUDA(cudaMalloc(&pl->partials, ncta * 4 * sizeof(double)));
        LQ_PLAN_CUDA(cudaMalloc(&pl->partials0, ncta * 2 * sizeof(double)));
        LQ_PLAN_CUDA(cudaMalloc(&pl->counter, sizeof(unsigned int)));
    }
    if (masked && (pl->sites_dirty || rebuild || pl->flags_seen != f.flags || pl->kind_seen != f.kind)) {
        const size_t nts = (size_t)pl->ntx * pl->nty * (g.Lz + 2);
        cudaFree(pl->tsum); pl->tsum = nullptr;
        LQ_PLAN_CUDA(cudaMalloc(&pl->tsum, nts));
        if (stored_F) {
            if (!pl->plain) LQ_PLAN_CUDA(cudaMalloc(&pl->plain, (size_t)g.NP));
            LQ_PLAN_CUDA(cudaMemsetAsync(pl->plain, 0, (size_t)g.NP, st));
            lq_launch_plain_map(g, f.flags, pl->plain, st);
            lq_launch_tile_summary(g, pl->plain, pl->tsum, TX, TY, pl->ntx, pl->nty, st);
            if (lq_fixup_build_list(g, f.flags, pl->plain, &pl->np_list, &pl->n_np, st) != 0) { err = "lq_sweep: building the non-plain site list failed"; return LQ_ERR_NOMEM; }
            cudaFree(pl->partials2); pl->partials2 = nullptr;
            LQ_PLAN_CUDA(cudaMalloc(&pl->partials2, (size_t)4 * lq_fixup_num_blocks(pl->n_np) * sizeof(double)));
            if (!pl->counter2) LQ_PLAN_CUDA(cudaMalloc(&pl->counter2, sizeof(unsigned int)));
            LQ_PLAN_CUDA(cudaMemsetAsync(pl->counter2, 0, sizeof(unsigned int), st));
        } else {
            if (!pl->bond) LQ_PLAN_CUDA(cudaMalloc(&pl->bond, (size_t)g.NP * sizeof(uint32_t)));
            LQ_PLAN_CUDA(cudaMemsetAsync(pl->bond, 0, (size_t)g.NP * sizeof(uint32_t), st));
            lq_launch_bond_map(g, f.flags, f.kind, pl->bond, st);
            lq_launch_tile_summary_bond(g, pl->bond, pl->tsum, TX, TY, pl->ntx, pl->nty, st);
        }
        *launches += 2;
        pl->sites_dirty = false;
        pl->flags_seen = f.flags;
        pl->kind_seen = f.kind;
    }
    LQ_PLAN_CUDA(cudaMemsetAsync(pl->counter, 0, sizeof(unsigned int), st));
    return LQ_OK;
}

// One sweep (+ its fix-up launch on masked stored-force lattices) reading buffers `in`, writing `in ^ 1`.
// phase 0: both launches; 1: the sweep only; 2: the fix-up only (sub-domains: the fix-up reads q' across the slab
// faces, so the neighbours' new boundary planes must arrive between the two).
// first: first sweep of a call on the recompute path with velocity Verlet.  defer: leave the partials to a
// cross-domain reduction (sub-domains) instead of advancing the schedule in the last CTA.
int lq_sweep_step(LqSweepPlan *pl, bool stored_F, const LqGeom &g, const LqPhys &ph, const LqFields &f, double *q[2],
                  double *v[2], double *F[2], int in, LqFireScalars *dsc, const LqFireConsts &fc, bool first, bool defer,
                  cudaStream_t st, std::string &err, int phase) {
    using C1 = Cfg<32, 16>;
    using C3 = Cfg<32, 16>;
    using C6 = Cfg<32, 8>;      // cubic term: see lq_sweep_prepare
    const bool three = lq_three(ph);
    const bool masked = f.flags != nullptr;
    const int out = in ^ 1;
    SweepArgs a;
    memset(&a, 0, sizeof(a));
    a.g = g; a.ph = ph; a.f = f; a.sc = dsc; a.fc = fc; a.partials = pl->partials; a.counter = pl->counter;
    a.plain = pl->plain; a.tsum = pl->tsum; a.bond = pl->bond; a.work = pl->work; a.ntx = pl->ntx; a.nty = pl->nty;
    a.partials0 = pl->partials0;
    a.defer_advance = (defer || (masked && stored_F)) ? 1 : 0;
    a.qo = q[out]; a.vo = v[out]; a.Fo = F[out];
    const int ncta = pl->n_items;
    cudaError_t e = cudaSuccess;
    if (phase == 2) { /* fix-up only: the sweep of this step has run (sub-domains exchange q' in between) */ }
    else if (!stored_F)
        e = lq_launch_sweep_rc(masked, first, ncta, pl->attr_rc, pl->mq[in], pl->mv[in], a, st);
    else if (three && (ph.L4 != 0.0 || ph.L6 != 0.0)) {
        const int xt = (ph.L4 != 0.0 ? 1 : 0) | (ph.L6 != 0.0 ? 2 : 0);
        if (xt == 1) e = masked ? launch<C3, true, true, 1>(pl, in, a, 5, st) : launch<C3, true, false, 1>(pl, in, a, 4, st);
        else if (xt == 2) e = masked ? launch<C6, true, true, 2>(pl, in, a, 7, st) : launch<C6, true, false, 2>(pl, in, a, 6, st);
        else e = masked ? launch<C6, true, true, 3>(pl, in, a, 9, st) : launch<C6, true, false, 3>(pl, in, a, 8, st);
    }
    else if (three) e = masked ? launch<C3, true, true>(pl, in, a, 3, st) : launch<C3, true, false>(pl, in, a, 2, st);
    else e = masked ? launch<C1, false, true>(pl, in, a, 1, st) : launch<C1, false, false>(pl, in, a, 0, st);
    if (e == cudaSuccess && masked && stored_F && phase != 1)
        e = lq_launch_fixup(three, g, ph, f, q[out], v[out], F[out], pl->np_list, pl->n_np, dsc, fc, pl->partials,
                            ncta, pl->partials2, pl->counter2, st, defer ? 1 : 0);
    if (e != cudaSuccess) { err = std::string("lq_sweep launch: ") + cudaGetErrorString(e); return LQ_ERR_CUDA; }
    return LQ_OK;
}

// partial-sum segments of the last sweep (for the cross-domain reduction): returns how many were written (<= 3)
int lq_sweep_segments(const LqSweepPlan *pl, bool stored_F, bool masked, bool first, LqPartialSeg seg[3]) {
    int n = 0;
    const int ncta = pl->n_items;
    seg[n++] = LqPartialSeg{pl->partials, ncta, 4};
    if (stored_F && masked) seg[n++] = LqPartialSeg{pl->partials2, lq_fixup_num_blocks(pl->n_np), 4};
    if (first) seg[n++] = LqPartialSeg{pl->partials0, ncta, 2};
    return n;
}

int lq_sweep_run(LqSweepPlan **planp, bool stored_F, const LqGeom &g, const LqPhys &ph, const LqFields &f, double *q[2],
                 double *v[2], double *F[2], int *cur, LqFireScalars *dsc, const LqFireConsts &fc, long max_steps,
                 cudaStream_t st, long *launches, long *sweeps, LqFireScalars *h, std::string &err, int rc_chunks) {
    int rc = lq_sweep_prepare(planp, stored_F, g, ph, f, q, v, F, st, launches, err, rc_chunks);
    if (rc != LQ_OK) return rc;
    LqSweepPlan *pl = *planp;
    const bool masked = f.flags != nullptr;
    const int cur0 = *cur;
    // Sweeps to enqueue and buffer flips per step taken.  Recompute path, velocity Verlet: the first sweep also
    // carries the stop test on the initial state, so `max_steps` sweeps (one even if max_steps == 0) and the live
    // buffer flips once per counted step.  Stored path: one extra leading sweep evaluates F(q_0) (all coefficients
    // 0); Euler variant (either path): one extra sweep because every sweep is [drift of the scheduled step |
    // force | kick of the next one].  Those flip once more than steps were counted.
    const bool extra = stored_F || fc.euler;
    const long total = extra ? max_steps + 1 : (max_steps > 0 ? max_steps : 1);
    const long chunk = fc.force_tol > 0.0 ? 100 : (1L << 30);
    long done = 0;
    while (done < total) {
        const long n = (total - done) < chunk ? (total - done) : chunk;
        for (long i = 0; i < n; ++i) {
            const int in = (int)((cur0 + done + i) & 1);
            rc = lq_sweep_step(pl, stored_F, g, ph, f, q, v, F, in, dsc, fc, !stored_F && !fc.euler && done + i == 0, false, st, err);
            if (rc != LQ_OK) return rc;
        }
        done += n;
        *launches += (masked && stored_F) ? 2 * n : n; *sweeps += n;
        if (fc.force_tol > 0.0) {
            LQ_PLAN_CUDA(cudaMemcpyAsync(h, dsc, sizeof(*h), cudaMemcpyDeviceToHost, st));
            LQ_PLAN_CUDA(cudaStreamSynchronize(st));
            if (h->converged) break;
        }
    }
    LQ_PLAN_CUDA(cudaMemcpyAsync(h, dsc, sizeof(*h), cudaMemcpyDeviceToHost, st));
    LQ_PLAN_CUDA(cudaStreamSynchronize(st));
    *cur = (int)((cur0 + h->step + (extra ? 1 : 0)) & 1);
    return LQ_OK;
}

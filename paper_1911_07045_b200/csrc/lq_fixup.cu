// lq_fixup.cu -- second kernel of a FIRE step on MASKED lattices (sm_100a).
//
// The fused sweeps (lq_sweep_rc.cu, lq_sweep.cu) evaluate only constant-weight stencils.  Simulated sites whose
// stencil weights depend on the geometry ("non-plain": boundary sites, sites next to them, anchored sites;
// a few per cent of a lattice with walls / colloids) are left for this kernel, which runs over a compacted,
// index-ordered list of them:  F' = general gather-form force (boundary-aware differences, PAPER.md:183;
// anchoring Eq. 14/15) evaluated on the q' the sweep has just written; vc' = v_k + dt/2 F'
// (the sweep left v_k in the velocity slot); F' is stored for these sites only, for the next step's lazy
// rescale.  Its last block then reduces the sweep's per-CTA partials and its own per-block partials in index
// order and advances the FIRE schedule (Algorithm 1) on the device.
#include "lq_sweep.cuh"
#include "lq_sweep_dev.cuh"
#include "lq_site.cuh"

#include <cub/device/device_select.cuh>
#include <thrust/iterator/counting_iterator.h>

namespace {
using namespace lqsw;

constexpr int FB = 128;   // threads per block

struct FixArgs {
    LqGeom g;
    LqPhys ph;
    LqFields f;
    const double *q;        // q' (output buffer of the sweep), ghost shell valid
    double *v, *F;          // velocity slot (holds v_k on entry) and force slot of the same buffer
    const int *list;
    int n;
    LqFireScalars *sc;
    LqFireConsts fc;
    const double *sweep_partials;
    int n_sweep;
    double *partials;
    unsigned int *counter;
    int defer;              // sub-domains: publish the partials only; the cross-domain reduction advances the schedule
};

#ifndef LQ_FIX_MINB
#define LQ_FIX_MINB 4
#endif
template <bool THREE>
__global__ void __launch_bounds__(FB, LQ_FIX_MINB) k_fixup(const FixArgs a) {
    const LqFireScalars sc = *a.sc;
    if (sc.converged) return;
    const int i = blockIdx.x * FB + threadIdx.x;
    const long long NP = a.g.NP;
    const double hdt = lq_step_coef(sc, a.fc).kick;
    double r[4] = {0.0, 0.0, 0.0, 0.0};
    if (i < a.n) {
        const long long p = a.list[i];
        const unsigned fl = a.f.flags[p];
        int kind = 0; double W = 0.0, n[3] = {0.0, 0.0, 0.0};
        if (a.f.kind != nullptr && (fl & 3u) == 1u) {
            kind = a.f.kind[p];
            if (kind != 0) { W = a.f.W[p]; n[0] = a.f.axis[p]; n[1] = a.f.axis[NP + p]; n[2] = a.f.axis[2 * NP + p]; }
        }
        lqs::GlobalAcc acc{a.q, a.f.flags, NP, a.g.sy, a.g.sz, p};
        double Fn[5], vn[5];
        lqs::site_force<THREE>(a.ph, acc, fl, kind, W, n, Fn);
#pragma unroll
        for (int c = 0; c < 5; ++c) {
            vn[c] = __fma_rn(hdt, Fn[c], a.v[c * NP + p]);
            r[0] = __fma_rn(Fn[c], vn[c], r[0]);
            r[1] = __fma_rn(Fn[c], Fn[c], r[1]);
            r[2] = __fma_rn(vn[c], vn[c], r[2]);
            r[3] = fmax(r[3], fabs(Fn[c]));
            a.v[c * NP + p] = vn[c];
            a.F[c * NP + p] = Fn[c];
        }
        const int x = (int)(p % a.g.Px) - LQ_XO, y = (int)((p / a.g.Px) % a.g.Py) - LQ_GH,
                  z = (int)(p / a.g.sz) - LQ_GH;
        const int shx = ghost_shift(x, a.g.Lx, a.g.gwx), shy = ghost_shift(y, a.g.Ly, LQ_GH),
                  shz = ghost_shift_z(z, a.g);
        if (shx | shy | shz) {
            for (int m = 1; m < 8; ++m) {
                if (((m & 1) && !shx) || ((m & 2) && !shy) || ((m & 4) && !shz)) continue;
                const long long pg = p + ((m & 1) ? shx : 0) + ((m & 2) ? shy * a.g.sy : 0) + ((m & 4) ? shz * a.g.sz : 0);
#pragma unroll
                for (int c = 0; c < 5; ++c) { a.v[c * NP + pg] = vn[c]; a.F[c * NP + pg] = Fn[c]; }
            }
        }
    }
    // block partials -> last block: all partials (sweep CTAs first, then fix-up blocks) in index order
    __shared__ double red[4 * (FB / 32)];
    __shared__ unsigned s_last;
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    constexpr int NW = FB / 32;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const double w = k < 3 ? warp_sum(r[k]) : warp_max(r[k]);
        if (lane == 0) red[k * NW + wid] = w;
    }
    __syncthreads();
    if (tid == 0) {
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            double t = red[k * NW];
            for (int w = 1; w < NW; ++w) t = k < 3 ? t + red[k * NW + w] : fmax(t, red[k * NW + w]);
            a.partials[4 * blockIdx.x + k] = t;
        }
        if (a.defer) s_last = 0u;
        else {
            __threadfence();
            s_last = atomicAdd(a.counter, 1u) == gridDim.x - 1 ? 1u : 0u;
        }
    }
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    double t[4] = {0.0, 0.0, 0.0, 0.0};
    for (int b = tid; b < a.n_sweep; b += FB) {
        t[0] += __ldcg(a.sweep_partials + 4 * b); t[1] += __ldcg(a.sweep_partials + 4 * b + 1);
        t[2] += __ldcg(a.sweep_partials + 4 * b + 2); t[3] = fmax(t[3], __ldcg(a.sweep_partials + 4 * b + 3));
    }
    for (int b = tid; b < (int)gridDim.x; b += FB) {
        t[0] += __ldcg(a.partials + 4 * b); t[1] += __ldcg(a.partials + 4 * b + 1);
        t[2] += __ldcg(a.partials + 4 * b + 2); t[3] = fmax(t[3], __ldcg(a.partials + 4 * b + 3));
    }
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const double w = k < 3 ? warp_sum(t[k]) : warp_max(t[k]);
        if (lane == 0) red[k * NW + wid] = w;
    }
    __syncthreads();
    if (tid == 0) {
        double tot[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            tot[k] = red[k * NW];
            for (int w = 1; w < NW; ++w) tot[k] = k < 3 ? tot[k] + red[k * NW + w] : fmax(tot[k], red[k * NW + w]);
        }
        LqFireScalars nx = sc;
        lq_fire_advance_any(nx, a.fc, tot);
        *a.sc = nx;
        *a.counter = 0u;
    }
}

// predicate for the list: interior site, simulated, not plain
struct NonPlainPred {
    LqGeom g;
    const uint8_t *flags, *plain;
    __device__ bool operator()(int p) const {
        const int x = p % g.Px - LQ_XO, y = (p / g.Px) % g.Py - LQ_GH, z = (int)(p / g.sz) - LQ_GH;
        if (x < 0 || x >= g.Lx || y < 0 || y >= g.Ly || z < 0 || z >= g.Lz) return false;
        return plain[p] == 0 && (flags[p] & 3u) != 2u;
    }
};

}  // namespace

// Build the index-ordered list of non-plain simulated sites.  *list is (re)allocated; *n receives the count.
int lq_fixup_build_list(const LqGeom &g, const uint8_t *flags, const uint8_t *plain, int **list, int *n,
                        cudaStream_t st) {
    int *d_n = nullptr, *d_out = nullptr;
    void *tmp = nullptr;
    size_t tmp_bytes = 0;
    if (cudaMalloc(&d_n, sizeof(int)) != cudaSuccess) return -1;
    // worst case every site is listed; count first with a null output to size the list exactly
    thrust::counting_iterator<int> it(0);
    NonPlainPred pred{g, flags, plain};
    if (cudaMalloc(&d_out, (size_t)g.N * sizeof(int)) != cudaSuccess) { cudaFree(d_n); return -1; }
    cub::DeviceSelect::If(nullptr, tmp_bytes, it, d_out, d_n, (int)g.NP, pred, st);
    if (cudaMalloc(&tmp, tmp_bytes) != cudaSuccess) { cudaFree(d_n); cudaFree(d_out); return -1; }
    cub::DeviceSelect::If(tmp, tmp_bytes, it, d_out, d_n, (int)g.NP, pred, st);
    int h = 0;
    cudaMemcpyAsync(&h, d_n, sizeof(int), cudaMemcpyDeviceToHost, st);
    cudaError_t e = cudaStreamSynchronize(st);
    cudaFree(tmp); cudaFree(d_n);
    if (e != cudaSuccess) { cudaFree(d_out); return -1; }
    // shrink to fit
    int *fit = nullptr;
    if (cudaMalloc(&fit, (size_t)(h > 0 ? h : 1) * sizeof(int)) != cudaSuccess) { cudaFree(d_out); return -1; }
    if (h > 0) cudaMemcpyAsync(fit, d_out, (size_t)h * sizeof(int), cudaMemcpyDeviceToDevice, st);
    cudaStreamSynchronize(st);
    cudaFree(d_out);
    cudaFree(*list);
    *list = fit; *n = h;
    return 0;
}

int lq_fixup_num_blocks(int n) { return n > 0 ? (n + FB - 1) / FB : 1; }

cudaError_t lq_launch_fixup(bool three, const LqGeom &g, const LqPhys &ph, const LqFields &f, const double *q,
                            double *v, double *F, const int *list, int n, LqFireScalars *sc, const LqFireConsts &fc,
                            const double *sweep_partials, int n_sweep, double *partials, unsigned int *counter,
                            cudaStream_t st, int defer) {
    FixArgs a{g, ph, f, q, v, F, list, n, sc, fc, sweep_partials, n_sweep, partials, counter, defer};
    const int nb = lq_fixup_num_blocks(n);
    if (three) k_fixup<true><<<nb, FB, 0, st>>>(a);
    else k_fixup<false><<<nb, FB, 0, st>>>(a);
    return cudaGetLastError();
}

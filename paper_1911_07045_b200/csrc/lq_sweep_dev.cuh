// lq_sweep_dev.cuh -- device helpers shared by the fused sweep kernels (TMA / mbarrier PTX wrappers,
// the drift formula, and the end-of-step reduction + on-device FIRE schedule).
#pragma once
#include "lq_internal.cuh"
#include <cuda.h>

namespace lqsw {

struct SweepArgs {
    LqGeom g;
    LqPhys ph;
    LqFields f;
    double *qo, *vo, *Fo;
    LqFireScalars *sc;
    LqFireConsts fc;
    double *partials;
    unsigned int *counter;
    const uint8_t *plain;   // stored-force sweep, masked lattices: per-site 'constant stencil weights' byte
    const uint8_t *tsum;    // per (plane, tile): tile + halo all plain
    int defer_advance;      // stored-force sweep on masked lattices: the fix-up kernel (lq_fixup.cu) finishes the step
    const int4 *work;       // work items (tile x, tile y, first plane, end plane), longest first; one per CTA
    int ntx, nty;           // tiles per row / column (indexing of tsum)
    // recompute sweep (lq_sweep_rc.cu)
    const uint32_t *bond;   // masked lattices: per-site bond code (LQ_BOND_*), ghost margin of 1 filled
    double *partials0;      // first sweep: per-CTA (|F(q_0)|^2, max|F_a(q_0)|) of the initial state
};

// ---------------------------------------------------------------- PTX wrappers (TMA + mbarrier)
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t *bar, int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_LOOP:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra WAIT_DONE;\n"
        "bra WAIT_LOOP;\n"
        "WAIT_DONE:\n"
        "}\n" ::"r"(smem_u32(bar)),
        "r"(parity)
        : "memory");
}
__device__ __forceinline__ void tma_load_4d(void *dst, const CUtensorMap *map, uint64_t *bar, int c0, int c1, int c2,
                                            int c3) {
    asm volatile(
        "cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6}], [%2];"
        ::"r"(smem_u32(dst)), "l"(map), "r"(smem_u32(bar)), "r"(c0), "r"(c1), "r"(c2), "r"(c3)
        : "memory");
}

// 4-byte global -> shared copy that bypasses the register file (LDGSTS); commit / wait by group
__device__ __forceinline__ void cp_async_4(void *dst, const void *src) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(smem_u32(dst)), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_but_one() { asm volatile("cp.async.wait_group 1;" ::: "memory"); }

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    return v;
}
__device__ __forceinline__ double warp_max(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_down_sync(0xffffffffu, v, o));
    return v;
}


// q' and v_k of one site from (q, vc, F): v_k = mix_a vc + (mix_b + dt/2) F ; q' = q + dt v_k.
// The SAME instruction sequence serves a CTA's own sites and the halo copies its neighbours compute,
// so every CTA sees bit-identical q'.
// ma == 0 (first step of a call, or after a P <= 0 reset) drops vc without reading its value, so a velocity
// buffer that was never written (or holds an earlier run's NaN) cannot leak in; likewise cF == 0 and F.
__device__ __forceinline__ void drift(double q, double vc, double F, double ma, double cF, double dt, double &vk,
                                      double &qn) {
    const double kF = cF == 0.0 ? 0.0 : cF * F;
    vk = ma == 0.0 ? kF : __fma_rn(ma, vc, kF);
    qn = __fma_rn(dt, vk, q);
}

// ghost-shell shift of coordinate i in a periodic dimension of length L, ghost width gw (0 if interior)
__device__ __forceinline__ int ghost_shift(int i, int L, int gw) { return i < gw ? L : (i >= L - gw ? -L : 0); }
// same along z: a sub-domain (g.zopen) has no periodic image in z, its z ghost planes are the neighbours'
__device__ __forceinline__ int ghost_shift_z(int k, const LqGeom &g) { return g.zopen ? 0 : ghost_shift(k, g.Lz, LQ_GH); }

// End of a sweep: block-reduce r = (P, FF, vv, Fmax) partials, publish them, and let the LAST CTA to finish
// reduce all CTAs' partials in index order (bitwise reproducible) and advance the FIRE schedule
// (Algorithm 1) in place.  red: >= 4*NT/32 doubles of shared memory.
// FIRST (recompute path, first sweep of a call): r0 = (|F(q_0)|^2, max|F_a(q_0)|) of the initial state is reduced
// the same way and decides Algorithm 1's stop test on the initial state (lq_fire_advance_first).
template <int NT, bool FIRST = false>
__device__ __forceinline__ void finish_step(const SweepArgs &a, const LqFireScalars &sc, const double r[4], double *red,
                                            const double *r0 = nullptr) {
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    constexpr int NW = NT / 32;
    __shared__ unsigned s_last;
    __shared__ double s_tot0[2];
    const unsigned ncta = gridDim.x * gridDim.y * gridDim.z;
    const unsigned cta = blockIdx.x + gridDim.x * (blockIdx.y + gridDim.y * blockIdx.z);
    if (FIRST) {
        const double w0 = warp_sum(r0[0]), w1 = warp_max(r0[1]);
        if (lane == 0) { red[wid] = w0; red[NW + wid] = w1; }
        __syncthreads();
        if (tid == 0) {
            double t0 = red[0], t1 = red[NW];
            for (int w = 1; w < NW; ++w) { t0 += red[w]; t1 = fmax(t1, red[NW + w]); }
            a.partials0[2 * cta] = t0; a.partials0[2 * cta + 1] = t1;
        }
        __syncthreads();
    }
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const double w = i < 3 ? warp_sum(r[i]) : warp_max(r[i]);
        if (lane == 0) red[i * NW + wid] = w;
    }
    __syncthreads();
    if (tid == 0) {
        double t[4];
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            t[i] = red[i * NW];
            for (int w = 1; w < NW; ++w) t[i] = i < 3 ? t[i] + red[i * NW + w] : fmax(t[i], red[i * NW + w]);
            a.partials[4 * cta + i] = t[i];
        }
        if (a.defer_advance) s_last = 0u;
        else {
            __threadfence();
            s_last = atomicAdd(a.counter, 1u) == ncta - 1 ? 1u : 0u;
        }
    }
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    if (FIRST) {
        double t0 = 0.0, t1 = 0.0;
        for (unsigned b = tid; b < ncta; b += NT) { t0 += __ldcg(a.partials0 + 2 * b); t1 = fmax(t1, __ldcg(a.partials0 + 2 * b + 1)); }
        t0 = warp_sum(t0); t1 = warp_max(t1);
        if (lane == 0) { red[wid] = t0; red[NW + wid] = t1; }
        __syncthreads();
        if (tid == 0) {
            double u0 = red[0], u1 = red[NW];
            for (int w = 1; w < NW; ++w) { u0 += red[w]; u1 = fmax(u1, red[NW + w]); }
            s_tot0[0] = u0; s_tot0[1] = u1;
        }
        __syncthreads();
    }
    double t[4] = {0.0, 0.0, 0.0, 0.0};
    for (unsigned b = tid; b < ncta; b += NT) {
        t[0] += __ldcg(a.partials + 4 * b); t[1] += __ldcg(a.partials + 4 * b + 1); t[2] += __ldcg(a.partials + 4 * b + 2);
        t[3] = fmax(t[3], __ldcg(a.partials + 4 * b + 3));
    }
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const double w = i < 3 ? warp_sum(t[i]) : warp_max(t[i]);
        if (lane == 0) red[i * NW + wid] = w;
    }
    __syncthreads();
    if (tid == 0) {
        double tot[4];
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            tot[i] = red[i * NW];
            for (int w = 1; w < NW; ++w) tot[i] = i < 3 ? tot[i] + red[i * NW + w] : fmax(tot[i], red[i * NW + w]);
        }
        LqFireScalars nx = sc;
        if (FIRST) lq_fire_advance_first(nx, a.fc, tot, s_tot0);
        else lq_fire_advance_any(nx, a.fc, tot);
        *a.sc = nx;
        *a.counter = 0u;
    }
}

}  // namespace lqsw

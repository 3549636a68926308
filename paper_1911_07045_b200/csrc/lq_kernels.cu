// lq_kernels.cu -- generic kernels: ghost refresh, site classification, force field,
// energy, and the unfused FIRE path (fire_path = 1).  One thread per lattice site, global
// loads through L1/L2.  These serve lq_set_sites / lq_forces / lq_energy and are the
// cross-check for the fused sweep (lq_sweep.cu), which is the product's hot path.
#include "lq_ctx.cuh"
#include "lq_internal.cuh"
#include "lq_site.cuh"

#include <mutex>

namespace {

constexpr int BX = 64, BY = 4;      // block shape for per-site kernels
constexpr int ZPER = 8;             // z planes per block

__device__ __forceinline__ int wrap(int i, int L) { return i < 0 ? i + L : (i >= L ? i - L : i); }

// ---- ghost shell refresh: every padded cell outside the interior copies its periodic image
template <typename T>
__global__ void k_fill_ghosts(LqGeom g, T *field, int ncomp) {
    const int px = blockIdx.x * blockDim.x + threadIdx.x;  // 0 .. Lx+2GH-1 -> x = px - GH
    const int py = blockIdx.y * blockDim.y + threadIdx.y;
    const int pz = blockIdx.z;
    if (px >= g.Lx + 2 * LQ_GH || py >= g.Py) return;
    const int x = px - LQ_GH, y = py - LQ_GH, z = pz - LQ_GH;
    // sub-domain (zopen): nothing wraps in z; every padded plane, its z ghost planes included, gets its x/y ghosts
    const bool zin = g.zopen || (z >= 0 && z < g.Lz);
    if (x >= 0 && x < g.Lx && y >= 0 && y < g.Ly && zin) return;
    const long long dst = g.pidx(x, y, z);
    const long long src = g.pidx(wrap(x, g.Lx), wrap(y, g.Ly), g.zopen ? z : wrap(z, g.Lz));
    for (int c = 0; c < ncomp; ++c) field[c * g.NP + dst] = field[c * g.NP + src];
}

// ---- classification (R8).  mask_p has its ghost shell filled.
__global__ void k_classify(LqGeom g, const uint8_t *__restrict__ mask_p, uint8_t *__restrict__ flags_p) {
    const int x = blockIdx.x * blockDim.x + threadIdx.x;
    const int y = blockIdx.y * blockDim.y + threadIdx.y;
    const int z = blockIdx.z;
    if (x >= g.Lx || y >= g.Ly) return;
    const long long p = g.pidx(x, y, z);
    const long long off[6] = {1, -1, g.sy, -g.sy, g.sz, -g.sz};
    unsigned f = 0, any_obj = 0;
#pragma unroll
    for (int b = 0; b < 6; ++b) {
        const unsigned sim = mask_p[p + off[b]] == 0;
        f |= sim << (2 + b);
        any_obj |= !sim;
    }
    const unsigned cls = mask_p[p] != 0 ? 2u : (any_obj ? 1u : 0u);
    flags_p[p] = (uint8_t)(f | cls);
}

// sub-domain classification: dense mask with a 3-plane margin (planes -3 .. Lz+2, periodic in x and y) -> packed
// flags on planes -2 .. Lz+1 (the full z ghost width), same bit layout as k_classify
__global__ void k_classify_ext(LqGeom g, const uint8_t *__restrict__ m, uint8_t *__restrict__ flags_p) {
    const int x = blockIdx.x * blockDim.x + threadIdx.x;
    const int y = blockIdx.y * blockDim.y + threadIdx.y;
    const int z = (int)blockIdx.z - LQ_GH;                   // -2 .. Lz+1
    if (x >= g.Lx || y >= g.Ly) return;
    auto at = [&](int xx, int yy, int zz) -> unsigned {
        return m[(size_t)wrap(xx, g.Lx) + (size_t)g.Lx * ((size_t)wrap(yy, g.Ly) + (size_t)g.Ly * (size_t)(zz + 3))];
    };
    const unsigned nb[6] = {at(x + 1, y, z), at(x - 1, y, z), at(x, y + 1, z), at(x, y - 1, z), at(x, y, z + 1), at(x, y, z - 1)};
    unsigned f = 0, any_obj = 0;
#pragma unroll
    for (int b = 0; b < 6; ++b) {
        const unsigned sim = nb[b] == 0;
        f |= sim << (2 + b);
        any_obj |= !sim;
    }
    const unsigned cls = at(x, y, z) != 0 ? 2u : (any_obj ? 1u : 0u);
    flags_p[g.pidx(x, y, z)] = (uint8_t)(f | cls);
}

__global__ void k_count_classes(LqGeom g, const uint8_t *__restrict__ flags_p, unsigned long long *counts) {
    const int x = blockIdx.x * blockDim.x + threadIdx.x;
    const int y = blockIdx.y * blockDim.y + threadIdx.y;
    const int z = blockIdx.z;
    __shared__ unsigned c[3];
    const int tid = threadIdx.y * blockDim.x + threadIdx.x;
    if (tid < 3) c[tid] = 0;
    __syncthreads();
    if (x < g.Lx && y < g.Ly) atomicAdd(&c[flags_p[g.pidx(x, y, z)] & 3u], 1u);
    __syncthreads();
    if (tid < 3 && c[tid]) atomicAdd(&counts[tid], (unsigned long long)c[tid]);
}

__global__ void k_check_u8_max(LqGeom g, const uint8_t *__restrict__ a, int maxval, int *bad) {
    const int x = blockIdx.x * blockDim.x + threadIdx.x;
    const int y = blockIdx.y * blockDim.y + threadIdx.y;
    const int z = blockIdx.z;
    if (x < g.Lx && y < g.Ly && a[g.pidx(x, y, z)] > maxval) *bad = 1;
}

// dense byte array: mode 0: any value > ref; mode 1: any value != ref
__global__ void k_check_dense_u8(const uint8_t *__restrict__ a, long long n, int ref, int mode, int *bad) {
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x)
        if (mode == 0 ? a[i] > ref : a[i] != ref) *bad = 1;
}

__device__ __forceinline__ void load_anchor(const LqFields &f, long long NP, long long p, unsigned fl, int &kind,
                                            double &W, double n[3]) {
    kind = 0; W = 0.0; n[0] = n[1] = n[2] = 0.0;
    if (f.kind != nullptr && (fl & 3u) == 1u) {
        kind = f.kind[p];
        if (kind != 0) { W = f.W[p]; n[0] = f.axis[p]; n[1] = f.axis[NP + p]; n[2] = f.axis[2 * NP + p]; }
    }
}

// ---- force field (lq_forces)
template <bool THREE>
__global__ void __launch_bounds__(BX * BY) k_forces(LqGeom g, LqPhys ph, LqFields f, const double *__restrict__ q,
                                                    double *__restrict__ F) {
    const int x = blockIdx.x * BX + threadIdx.x;
    const int y = blockIdx.y * BY + threadIdx.y;
    if (x >= g.Lx || y >= g.Ly) return;
    for (int z = blockIdx.z * ZPER; z < min(g.Lz, (int)(blockIdx.z + 1) * ZPER); ++z) {
        const long long p = g.pidx(x, y, z);
        const unsigned fl = f.flags ? f.flags[p] : 0xFCu;
        double Fs[5] = {0, 0, 0, 0, 0};
        if ((fl & 3u) != 2u) {
            int kind; double W, n[3];
            load_anchor(f, g.NP, p, fl, kind, W, n);
            lqs::GlobalAcc acc{q, f.flags, g.NP, g.sy, g.sz, p};
            lqs::site_force<THREE>(ph, acc, fl, kind, W, n, Fs);
        }
#pragma unroll
        for (int c = 0; c < 5; ++c) F[c * g.NP + p] = Fs[c];
    }
}

// ---- block reduction helpers (fixed order -> bitwise reproducible)
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

template <int NV, int NT>
__device__ __forceinline__ void block_reduce(double (&val)[NV], int nsum, double *out) {
    // first nsum entries are summed, the rest are max-reduced; result written by thread 0
    __shared__ double sm[NV][NT / 32];
    const int tid = threadIdx.y * blockDim.x + threadIdx.x;
    const int lane = tid & 31, wid = tid >> 5;
#pragma unroll
    for (int i = 0; i < NV; ++i) {
        const double r = i < nsum ? warp_sum(val[i]) : warp_max(val[i]);
        if (lane == 0) sm[i][wid] = r;
    }
    __syncthreads();
    if (tid == 0) {
#pragma unroll
        for (int i = 0; i < NV; ++i) {
            double r = sm[i][0];
            for (int w = 1; w < NT / 32; ++w) r = i < nsum ? r + sm[i][w] : fmax(r, sm[i][w]);
            out[i] = r;
        }
    }
}

// ---- energy
template <bool THREE>
__global__ void __launch_bounds__(BX * BY) k_energy(LqGeom g, LqPhys ph, LqFields f, const double *__restrict__ q,
                                                    double *__restrict__ partials) {
    const int x = blockIdx.x * BX + threadIdx.x;
    const int y = blockIdx.y * BY + threadIdx.y;
    double acc3[3] = {0, 0, 0};
    if (x < g.Lx && y < g.Ly) {
        for (int z = blockIdx.z * ZPER; z < min(g.Lz, (int)(blockIdx.z + 1) * ZPER); ++z) {
            const long long p = g.pidx(x, y, z);
            const unsigned fl = f.flags ? f.flags[p] : 0xFCu;
            if ((fl & 3u) == 2u) continue;
            int kind; double W, n[3], t[3];
            load_anchor(f, g.NP, p, fl, kind, W, n);
            lqs::GlobalAcc acc{q, f.flags, g.NP, g.sy, g.sz, p};
            lqs::site_energy<THREE>(ph, acc, fl, kind, W, n, t);
            acc3[0] += t[0]; acc3[1] += t[1]; acc3[2] += t[2];
        }
    }
    const long long b = blockIdx.x + (long long)gridDim.x * (blockIdx.y + (long long)gridDim.y * blockIdx.z);
    block_reduce<3, BX * BY>(acc3, 3, partials + 3 * b);
}

// final reduce: one block, fixed order, Neumaier-compensated per thread then tree
template <int NV>
__global__ void __launch_bounds__(256) k_final_sum(const double *__restrict__ partials, long long nblocks,
                                                   double *__restrict__ out) {
    double s[NV], c[NV];
#pragma unroll
    for (int i = 0; i < NV; ++i) { s[i] = 0.0; c[i] = 0.0; }
    for (long long b = threadIdx.x; b < nblocks; b += 256) {
#pragma unroll
        for (int i = 0; i < NV; ++i) {
            const double v = partials[NV * b + i];
            const double t = s[i] + v;
            c[i] += fabs(s[i]) >= fabs(v) ? (s[i] - t) + v : (v - t) + s[i];
            s[i] = t;
        }
    }
#pragma unroll
    for (int i = 0; i < NV; ++i) s[i] += c[i];
    block_reduce<NV, 256>(s, NV, out);
}

// ---- unfused FIRE (fire_path = 1)  Algorithm 1
// drift: v <- mix_a v + mix_b F (the rescale decided by the previous step's reductions);
//        v += dt/2 F; q += dt v          (simulated sites only)
__global__ void __launch_bounds__(BX * BY) k_fire1_drift(LqGeom g, LqFields f, double *__restrict__ q,
                                                         double *__restrict__ v, const double *__restrict__ F,
                                                         const LqFireScalars *__restrict__ sc, int euler) {
    if (sc->converged) return;
    const int x = blockIdx.x * BX + threadIdx.x;
    const int y = blockIdx.y * BY + threadIdx.y;
    if (x >= g.Lx || y >= g.Ly) return;
    const double dt = sc->dt, ma = sc->mix_a, mb = sc->mix_b;
    for (int z = blockIdx.z * ZPER; z < min(g.Lz, (int)(blockIdx.z + 1) * ZPER); ++z) {
        const long long p = g.pidx(x, y, z);
        if (f.flags && (f.flags[p] & 3u) == 2u) continue;
#pragma unroll
        for (int c = 0; c < 5; ++c) {
            const long long i = c * g.NP + p;
            const double Fc = F[i];
            double vc = ma * v[i] + mb * Fc;
            if (!euler) vc += 0.5 * dt * Fc;
            v[i] = vc;
            q[i] += (euler ? sc->dt_prev : dt) * vc;
        }
    }
}

// force + second half kick + partial reductions of P = F.v, |F|^2, |v|^2, max|F_a|
template <bool THREE>
__global__ void __launch_bounds__(BX * BY) k_fire1_force(LqGeom g, LqPhys ph, LqFields f,
                                                         const double *__restrict__ q, double *__restrict__ v,
                                                         double *__restrict__ F, const LqFireScalars *__restrict__ sc,
                                                         double *__restrict__ partials, long long euler_max) {
    if (sc->converged) return;
    const int x = blockIdx.x * BX + threadIdx.x;
    const int y = blockIdx.y * BY + threadIdx.y;
    // velocity Verlet: second half kick; Euler variant: the full kick of the next step, none once the budget is spent
    const double hdt = euler_max < 0 ? 0.5 * sc->dt : (sc->step < euler_max ? sc->dt : 0.0);
    double r[4] = {0, 0, 0, 0};
    if (x < g.Lx && y < g.Ly) {
        for (int z = blockIdx.z * ZPER; z < min(g.Lz, (int)(blockIdx.z + 1) * ZPER); ++z) {
            const long long p = g.pidx(x, y, z);
            const unsigned fl = f.flags ? f.flags[p] : 0xFCu;
            double Fs[5] = {0, 0, 0, 0, 0};
            const bool sim = (fl & 3u) != 2u;
            if (sim) {
                int kind; double W, n[3];
                load_anchor(f, g.NP, p, fl, kind, W, n);
                lqs::GlobalAcc acc{q, f.flags, g.NP, g.sy, g.sz, p};
                lqs::site_force<THREE>(ph, acc, fl, kind, W, n, Fs);
            }
#pragma unroll
            for (int c = 0; c < 5; ++c) {
                const long long i = c * g.NP + p;
                F[i] = Fs[c];
                if (sim) {
                    const double vc = v[i] + hdt * Fs[c];
                    v[i] = vc;
                    r[0] += Fs[c] * vc; r[1] += Fs[c] * Fs[c]; r[2] += vc * vc; r[3] = fmax(r[3], fabs(Fs[c]));
                }
            }
        }
    }
    const long long b = blockIdx.x + (long long)gridDim.x * (blockIdx.y + (long long)gridDim.y * blockIdx.z);
    block_reduce<4, BX * BY>(r, 3, partials + 4 * b);
}

// One block: reduce the per-block partials in a fixed order, then advance the FIRE schedule.
// first != 0: this is the initial force evaluation (step 0): only the convergence test applies.
__global__ void __launch_bounds__(256) k_fire_update(const double *__restrict__ partials, int nblocks,
                                                     LqFireScalars *sc, LqFireConsts fc, int first) {
    if (sc->converged) return;
    double s[4] = {0, 0, 0, 0};
    for (int b = threadIdx.x; b < nblocks; b += 256) {
        s[0] += partials[4 * b]; s[1] += partials[4 * b + 1]; s[2] += partials[4 * b + 2];
        s[3] = fmax(s[3], partials[4 * b + 3]);
    }
    __shared__ double tot[4];
    block_reduce<4, 256>(s, 3, tot);
    __syncthreads();
    if (threadIdx.x != 0) return;
    LqFireScalars t = *sc;
    if (first == 2) lq_fire_advance_euler(t, fc, tot);
    else lq_fire_advance(t, fc, tot, first);
    *sc = t;
}

// Cross-domain reduction of one step ("one tiny all-reduce"): the per-CTA partials of
// every sub-domain's sweep (and fix-up) in a FIXED order -> tot6 = (P, FF, vv, Fmax, FF0, Fmax0).  Segments of width 4
// feed the first four, segments of width 2 (the first sweep's initial-state partials) the last two.
__global__ void __launch_bounds__(256) k_reduce_partials(const LqPartialSeg *__restrict__ seg, int nseg,
                                                         double *__restrict__ tot6) {
    double s[6] = {0, 0, 0, 0, 0, 0};
    for (int i = 0; i < nseg; ++i) {
        const LqPartialSeg sg = seg[i];
        if (sg.width == 4) {
            for (int b = threadIdx.x; b < sg.n; b += 256) {
                s[0] += sg.p[4 * b]; s[1] += sg.p[4 * b + 1]; s[2] += sg.p[4 * b + 2]; s[3] = fmax(s[3], sg.p[4 * b + 3]);
            }
        } else {
            for (int b = threadIdx.x; b < sg.n; b += 256) { s[4] += sg.p[2 * b]; s[5] = fmax(s[5], sg.p[2 * b + 1]); }
        }
    }
    // order: sums first (block_reduce sums the first nsum entries, max-reduces the rest)
    double r[6] = {s[0], s[1], s[2], s[4], s[3], s[5]};
    __shared__ double out[6];
    block_reduce<6, 256>(r, 4, out);
    __syncthreads();
    if (threadIdx.x == 0) {
        tot6[0] = out[0]; tot6[1] = out[1]; tot6[2] = out[2]; tot6[3] = out[4]; tot6[4] = out[3]; tot6[5] = out[5];
    }
}

// tot: nrank x 6 (one row per rank / sub-domain group, combined in rank order) -> the same schedule update in every
// sub-domain's scalars.  first: the sweep just reduced was the first of the call (recompute path, velocity Verlet).
__global__ void k_advance(const double *__restrict__ tot, int nrank, LqFireScalars *const *__restrict__ scs, int nsc,
                          LqFireConsts fc, int first) {
    if (threadIdx.x != 0 || blockIdx.x != 0) return;
    double t[4] = {0, 0, 0, 0}, t0[2] = {0, 0};
    for (int r = 0; r < nrank; ++r) {
        t[0] += tot[6 * r]; t[1] += tot[6 * r + 1]; t[2] += tot[6 * r + 2]; t[3] = fmax(t[3], tot[6 * r + 3]);
        t0[0] += tot[6 * r + 4]; t0[1] = fmax(t0[1], tot[6 * r + 5]);
    }
    LqFireScalars nx = *scs[0];
    if (nx.converged) return;
    if (first) lq_fire_advance_first(nx, fc, t, t0);
    else lq_fire_advance_any(nx, fc, t);
    for (int i = 0; i < nsc; ++i) *scs[i] = nx;
}

__global__ void k_zero_object_sites(LqGeom g, const uint8_t *__restrict__ flags, double *__restrict__ field) {
    const int x = blockIdx.x * blockDim.x + threadIdx.x;
    const int y = blockIdx.y * blockDim.y + threadIdx.y;
    const int z = blockIdx.z;
    if (x >= g.Lx || y >= g.Ly) return;
    const long long p = g.pidx(x, y, z);
    if ((flags[p] & 3u) == 2u)
        for (int c = 0; c < 5; ++c) field[c * g.NP + p] = 0.0;
}

// plain[p] = 1 iff the site is bulk with all 6 neighbours simulated AND each of its 6 neighbours also has all
// 6 of its neighbours simulated (constant stencil weights).  Computed on the interior plus
// a one-site ghost margin (flags carry a 2-wide ghost shell).
__global__ void k_plain_map(LqGeom g, const uint8_t *__restrict__ flags, uint8_t *__restrict__ plain) {
    const int x = (int)(blockIdx.x * blockDim.x + threadIdx.x) - 1;
    const int y = (int)(blockIdx.y * blockDim.y + threadIdx.y) - 1;
    const int z = (int)blockIdx.z - 1;
    if (x > g.Lx || y > g.Ly) return;
    const long long p = g.pidx(x, y, z);
    const bool ok = flags[p] == 0xFCu && (flags[p + 1] >> 2) == 0x3Fu && (flags[p - 1] >> 2) == 0x3Fu &&
                    (flags[p + g.sy] >> 2) == 0x3Fu && (flags[p - g.sy] >> 2) == 0x3Fu &&
                    (flags[p + g.sz] >> 2) == 0x3Fu && (flags[p - g.sz] >> 2) == 0x3Fu;
    plain[p] = ok ? 1 : ((flags[p] & 3u) == 2u ? 2 : 0);   // 1 plain, 0 non-plain simulated, 2 object
}

// Bond codes of the one-constant masked sweep (lq_internal.cuh LQ_BOND_*): per direction the weight
// a^s_k(x) [w_k(x) + w_k(x + s k)] of the gather-form force, from the flag bytes
// of the site and its six neighbours.  Interior plus a one-site ghost margin (flags carry a 2-wide ghost shell).
__global__ void k_bond_map(LqGeom g, const uint8_t *__restrict__ flags, const uint8_t *__restrict__ kind,
                           uint32_t *__restrict__ bond) {
    const int x = (int)(blockIdx.x * blockDim.x + threadIdx.x) - 1;
    const int y = (int)(blockIdx.y * blockDim.y + threadIdx.y) - 1;
    const int z = (int)blockIdx.z - 1;
    if (x > g.Lx || y > g.Ly) return;
    const long long p = g.pidx(x, y, z);
    const unsigned fl = flags[p];
    unsigned code = 0;
    if ((fl & 3u) == 2u) code = LQ_BOND_OBJECT;
    else {
        const long long off[6] = {1, -1, g.sy, -g.sy, g.sz, -g.sz};
#pragma unroll
        for (int d = 0; d < 6; ++d) {
            if (!((fl >> (2 + d)) & 1u)) continue;
            const int k = d >> 1;
            const double w = lqs::w_axis(fl, k) + lqs::w_axis(flags[p + off[d]], k);     // 1, 3/2 or 2
            code |= (w == 1.0 ? 1u : (w == 1.5 ? 2u : 3u)) << (2 * d);
        }
        if ((fl & 3u) == 1u && kind != nullptr && kind[p] != 0) code |= LQ_BOND_ANCH;
    }
    bond[p] = (uint32_t)code;
}

// tsum[(z+1)][by][bx] = 1 iff every site of tile (bx, by) plus its one-site halo is plain at plane z (z = -1 .. Lz)
template <typename T>
__global__ void k_tile_summary(LqGeom g, const T *__restrict__ plain, unsigned plain_value, uint8_t *__restrict__ tsum,
                               int TX, int TY) {
    const int bx = blockIdx.x, by = blockIdx.y, z = (int)blockIdx.z - 1;
    int ok = 1;
    for (int i = threadIdx.x; i < (TX + 2) * (TY + 2); i += blockDim.x) {
        const int x = bx * TX - 1 + i % (TX + 2), y = by * TY - 1 + i / (TX + 2);
        if (x <= g.Lx && y <= g.Ly && (unsigned)plain[g.pidx(x, y, z)] != plain_value) ok = 0;
    }
    ok = __syncthreads_and(ok);
    if (threadIdx.x == 0) tsum[((size_t)(z + 1) * gridDim.y + by) * gridDim.x + bx] = (uint8_t)ok;
}

inline dim3 site_grid(const LqGeom &g) {
    return dim3((g.Lx + BX - 1) / BX, (g.Ly + BY - 1) / BY, (g.Lz + ZPER - 1) / ZPER);
}
inline dim3 plane_grid(const LqGeom &g) { return dim3((g.Lx + BX - 1) / BX, (g.Ly + BY - 1) / BY, g.Lz); }

}  // namespace

// fp64 FMA microbenchmark (the secondary roof of SURVEY 8(d)): 16 independent dependent-FMA chains per thread, no
// memory traffic; returns measured TFLOP/s (2 flop per FMA), < 0 on error.  Behind lq_get_info("fp64_fma_tflops").
namespace {
__global__ void __launch_bounds__(512) k_fp64_fma(double *out, int iters, double b, double c) {
    double a[16];
#pragma unroll
    for (int j = 0; j < 16; ++j) a[j] = 1.0 + 1e-3 * (double)(threadIdx.x + j);
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int j = 0; j < 16; ++j) a[j] = __fma_rn(a[j], b, c);
    }
    double s = 0.0;
#pragma unroll
    for (int j = 0; j < 16; ++j) s += a[j];
    out[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = s;
}
}  // namespace
double lq_measure_fp64_fma(int device, cudaStream_t st) {
    int nsm = 148;
    cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, device);
    const int nblk = 4 * nsm, nt = 512, iters = 1 << 14;
    double *out = nullptr;
    cudaEvent_t e0, e1;
    if (cudaMalloc(&out, (size_t)nblk * nt * sizeof(double)) != cudaSuccess) return -1.0;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    k_fp64_fma<<<nblk, nt, 0, st>>>(out, 256, 0.999999, 1e-7);          // warm-up
    float best = 0.f;
    for (int rep = 0; rep < 3; ++rep) {
        cudaEventRecord(e0, st);
        k_fp64_fma<<<nblk, nt, 0, st>>>(out, iters, 0.999999, 1e-7);
        cudaEventRecord(e1, st);
        cudaEventSynchronize(e1);
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        if (best == 0.f || ms < best) best = ms;
    }
    const cudaError_t err = cudaGetLastError();
    cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(out);
    if (err != cudaSuccess || best <= 0.f) return -1.0;
    return 2.0 * 16.0 * (double)iters * (double)nblk * nt / (best * 1e-3) / 1e12;
}

void lq_launch_fill_ghosts_f64(const LqGeom &g, double *field, int ncomp, cudaStream_t st) {
    dim3 b(64, 4), gr((g.Lx + 2 * LQ_GH + 63) / 64, (g.Py + 3) / 4, g.Pz);
    k_fill_ghosts<double><<<gr, b, 0, st>>>(g, field, ncomp);
}
void lq_launch_fill_ghosts_u8(const LqGeom &g, uint8_t *field, cudaStream_t st) {
    dim3 b(64, 4), gr((g.Lx + 2 * LQ_GH + 63) / 64, (g.Py + 3) / 4, g.Pz);
    k_fill_ghosts<uint8_t><<<gr, b, 0, st>>>(g, field, 1);
}
void lq_launch_classify(const LqGeom &g, const uint8_t *mask_p, uint8_t *flags_p, cudaStream_t st) {
    k_classify<<<plane_grid(g), dim3(BX, BY), 0, st>>>(g, mask_p, flags_p);
}
void lq_launch_classify_ext(const LqGeom &g, const uint8_t *mask_ext, uint8_t *flags_p, cudaStream_t st) {
    k_classify_ext<<<dim3((g.Lx + BX - 1) / BX, (g.Ly + BY - 1) / BY, g.Pz), dim3(BX, BY), 0, st>>>(g, mask_ext, flags_p);
}
void lq_launch_count_classes(const LqGeom &g, const uint8_t *flags_p, unsigned long long *counts3, cudaStream_t st) {
    k_count_classes<<<plane_grid(g), dim3(BX, BY), 0, st>>>(g, flags_p, counts3);
}
void lq_launch_check_u8_max(const LqGeom &g, const uint8_t *arr_p, int maxval, int *bad, cudaStream_t st) {
    k_check_u8_max<<<plane_grid(g), dim3(BX, BY), 0, st>>>(g, arr_p, maxval, bad);
}
void lq_launch_check_dense_u8_max(const uint8_t *a, long long n, int maxval, int *bad, cudaStream_t st) {
    k_check_dense_u8<<<148 * 4, 256, 0, st>>>(a, n, maxval, 0, bad);
}
void lq_launch_check_dense_u8_ne(const uint8_t *a, long long n, int value, int *bad, cudaStream_t st) {
    k_check_dense_u8<<<148 * 4, 256, 0, st>>>(a, n, value, 1, bad);
}
void lq_launch_forces(const LqGeom &g, const LqPhys &ph, const LqFields &f, const double *q, double *F,
                      cudaStream_t st) {
    if (lq_three(ph)) k_forces<true><<<site_grid(g), dim3(BX, BY), 0, st>>>(g, ph, f, q, F);
    else k_forces<false><<<site_grid(g), dim3(BX, BY), 0, st>>>(g, ph, f, q, F);
}
int lq_energy_num_blocks(const LqGeom &g) {
    dim3 gr = site_grid(g);
    return (int)(gr.x * gr.y * gr.z);
}
void lq_launch_energy(const LqGeom &g, const LqPhys &ph, const LqFields &f, const double *q, double *partials,
                      double *out3, cudaStream_t st) {
    if (lq_three(ph)) k_energy<true><<<site_grid(g), dim3(BX, BY), 0, st>>>(g, ph, f, q, partials);
    else k_energy<false><<<site_grid(g), dim3(BX, BY), 0, st>>>(g, ph, f, q, partials);
    k_final_sum<3><<<1, 256, 0, st>>>(partials, lq_energy_num_blocks(g), out3);
}
int lq_fire1_num_blocks(const LqGeom &g) { return lq_energy_num_blocks(g); }
void lq_launch_fire1_drift(const LqGeom &g, const LqFields &f, double *q, double *v, const double *F,
                           const LqFireScalars *sc, cudaStream_t st, int euler) {
    k_fire1_drift<<<site_grid(g), dim3(BX, BY), 0, st>>>(g, f, q, v, F, sc, euler);
}
void lq_launch_fire1_force(const LqGeom &g, const LqPhys &ph, const LqFields &f, const double *q, double *v,
                           double *F, const LqFireScalars *sc, double *partials, cudaStream_t st,
                           long long euler_max) {
    if (lq_three(ph))
        k_fire1_force<true><<<site_grid(g), dim3(BX, BY), 0, st>>>(g, ph, f, q, v, F, sc, partials, euler_max);
    else
        k_fire1_force<false><<<site_grid(g), dim3(BX, BY), 0, st>>>(g, ph, f, q, v, F, sc, partials, euler_max);
}
void lq_launch_fire_update(const double *partials, int nblocks, LqFireScalars *sc, LqFireConsts fc, int first,
                           cudaStream_t st) {
    k_fire_update<<<1, 256, 0, st>>>(partials, nblocks, sc, fc, first);
}
void lq_launch_reduce_partials(const LqPartialSeg *seg_dev, int nseg, double *tot6, cudaStream_t st) {
    k_reduce_partials<<<1, 256, 0, st>>>(seg_dev, nseg, tot6);
}
void lq_launch_advance(const double *tot, int nrank, LqFireScalars *const *sc_dev, int nsc, LqFireConsts fc, int first,
                       cudaStream_t st) {
    k_advance<<<1, 32, 0, st>>>(tot, nrank, sc_dev, nsc, fc, first);
}
void lq_launch_zero_object_sites(const LqGeom &g, const uint8_t *flags, double *field, cudaStream_t st) {
    k_zero_object_sites<<<plane_grid(g), dim3(BX, BY), 0, st>>>(g, flags, field);
}

// out = a v + b F over a whole padded 5-component field (lq_get_velocity: the FIRE rescale that the fused sweeps apply
// lazily, Algorithm 1 "rescale velocity")
__global__ void k_axpby(long long n, double a, const double *__restrict__ v, double b, const double *__restrict__ F,
                        double *__restrict__ out) {
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x)
        out[i] = a * v[i] + b * F[i];
}
void lq_launch_axpby(long long n, double a, const double *v, double b, const double *F, double *out, cudaStream_t st) {
    k_axpby<<<148 * 8, 256, 0, st>>>(n, a, v, b, F, out);
}

void lq_launch_plain_map(const LqGeom &g, const uint8_t *flags, uint8_t *plain, cudaStream_t st) {
    dim3 b(64, 4), gr((g.Lx + 2 + 63) / 64, (g.Ly + 2 + 3) / 4, g.Lz + 2);
    k_plain_map<<<gr, b, 0, st>>>(g, flags, plain);
}
void lq_launch_tile_summary(const LqGeom &g, const uint8_t *plain, uint8_t *tsum, int TX, int TY, int ntx, int nty,
                            cudaStream_t st) {
    k_tile_summary<uint8_t><<<dim3(ntx, nty, g.Lz + 2), 128, 0, st>>>(g, plain, 1u, tsum, TX, TY);
}
void lq_launch_bond_map(const LqGeom &g, const uint8_t *flags, const uint8_t *kind, uint32_t *bond, cudaStream_t st) {
    dim3 b(64, 4), gr((g.Lx + 2 + 63) / 64, (g.Ly + 2 + 3) / 4, g.Lz + 2);
    k_bond_map<<<gr, b, 0, st>>>(g, flags, kind, bond);
}
void lq_launch_tile_summary_bond(const LqGeom &g, const uint32_t *bond, uint8_t *tsum, int TX, int TY, int ntx, int nty,
                                 cudaStream_t st) {
    k_tile_summary<uint32_t><<<dim3(ntx, nty, g.Lz + 2), 128, 0, st>>>(g, bond, LQ_BOND_PLAIN, tsum, TX, TY);
}

// ---- lq_energy_terms_noalloc (include/lq.h): the energy pass of lq_energy_terms with its per-block partial sums in a
// static device array instead of a cudaMalloc'ed buffer.  Same two kernels, same launch shape, same summation order,
// so the three numbers are bit-identical to lq_energy_terms'.
namespace {

constexpr int LQ_NOALLOC_MAX_BLOCKS = 65536;   // k_energy blocks (64 x 4 x 8 sites each): 512^3 needs exactly this many

// 3 partial sums per block, then 3 doubles that stage the result for a host caller: 1.5 MiB of every GPU that loads
// liblq.so, held until the process exits.  Shared by all contexts and all calls.
static __device__ __align__(256) double g_noalloc_scratch[3 * LQ_NOALLOC_MAX_BLOCKS + 3];

constexpr int LQ_NOALLOC_MAX_DEVICES = 64;
double *g_noalloc_ptr[LQ_NOALLOC_MAX_DEVICES];  // device address of g_noalloc_scratch, by device ordinal (0 = not asked yet)
std::mutex g_noalloc_mu;

// In host code `g_noalloc_scratch` is only a handle for the runtime, not an address a kernel may dereference, and each
// device has its own copy of the array: ask the runtime for the address on the device that is current (the caller's
// DeviceGuard made that the context's device), once per device, and hand that pointer to the kernels.
cudaError_t noalloc_scratch(int device, double **out) {
    if (device < 0 || device >= LQ_NOALLOC_MAX_DEVICES) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_noalloc_mu);
    if (!g_noalloc_ptr[device]) {
        void *addr = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(&addr, g_noalloc_scratch);
        if (e != cudaSuccess) return e;
        g_noalloc_ptr[device] = static_cast<double *>(addr);
    }
    *out = g_noalloc_ptr[device];
    return cudaSuccess;
}

}  // namespace

extern "C" int lq_energy_terms_noalloc(lq_ctx *c, double *terms, int where) {
    if (!c) return LQ_ERR_ARG;
    DeviceGuard dg(c);
    if (!terms || bad_where(where)) return fail(c, LQ_ERR_ARG, "lq_energy_terms_noalloc: bad argument");
    const long long nblk = lq_energy_num_blocks(c->g);
    if (nblk > LQ_NOALLOC_MAX_BLOCKS)
        return fail(c, LQ_ERR_ARG, "lq_energy_terms_noalloc: this lattice needs " + std::to_string(nblk) +
                                       " reduction blocks (ceil(Lx/64) * ceil(Ly/4) * ceil(Lz/8)) but the static scratch "
                                       "array holds " + std::to_string(LQ_NOALLOC_MAX_BLOCKS) +
                                       "; use lq_energy_terms, which allocates");
    if (!c->has_Q) return fail(c, LQ_ERR_STATE, "lq_energy_terms_noalloc: no Q has been set");
    double *scratch = nullptr;
    LQ_CUDA(c, noalloc_scratch(c->device, &scratch));
    // nothing has to be cleared between calls: every block overwrites its own three slots and the final sum reads
    // exactly the nblk slots this launch wrote
    double *out3 = where == LQ_DEVICE ? terms : scratch + 3 * LQ_NOALLOC_MAX_BLOCKS;
    const LqFields f = fields_of(c);
    if (lq_three(c->ph)) k_energy<true><<<site_grid(c->g), dim3(BX, BY), 0, c->stream>>>(c->g, c->ph, f, c->q[c->cur], scratch);
    else k_energy<false><<<site_grid(c->g), dim3(BX, BY), 0, c->stream>>>(c->g, c->ph, f, c->q[c->cur], scratch);
    k_final_sum<3><<<1, 256, 0, c->stream>>>(scratch, nblk, out3);
    LQ_CUDA(c, cudaGetLastError());
    if (where == LQ_HOST) {
        LQ_CUDA(c, cudaMemcpyAsync(terms, out3, 3 * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
        LQ_CUDA(c, cudaStreamSynchronize(c->stream));
    }
    return LQ_OK;
}

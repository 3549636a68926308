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
    const int shx = ghost_shift(x, g.Lx, LQ_GH), shy = ghost_shift(y, g.Ly, LQ_GH), shz = ghost_shift(z, g.Lz, LQ_GH);
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

}  // namespace

struct LqDescentPlan {
    double *partials = nullptr;
    size_t cap = 0;
    unsigned int *counter = nullptr;
};

void lq_descent_destroy(LqDescentPlan *p) {
    if (!p) return;
    cudaFree(p->partials);
    cudaFree(p->counter);
    delete p;
}

// Runs up to max_steps steps, one launch per step (two on masked one-constant lattices once the sweep exists).
// buf[0] holds q_0 with a valid ghost shell; nbuf = 2 (GD) or 3 (Nesterov) rotating buffers.  On return *final
// is the index of the buffer that holds the last iterate and *h the scalars.
int lq_descent_run(LqDescentPlan **planp, int method, const LqGeom &g, const LqPhys &ph, const LqFields &f,
                   double *const *buf, int nbuf, int *final, LqFireScalars *dsc, double eta, double mu,
                   double force_tol, long max_steps, cudaStream_t st, long *launches, LqFireScalars *h,
                   std::string &err) {
    LqDescentPlan *pl = *planp;
    if (!pl) { pl = new LqDescentPlan(); *planp = pl; }
    const bool three = ph.L2 != 0.0 || ph.L3 != 0.0;
    const bool nest = method == LQ_MIN_NESTEROV;
    const unsigned nblk = (unsigned)((g.N + DB - 1) / DB);
    if (pl->cap < (size_t)2 * nblk) {
        cudaFree(pl->partials); pl->partials = nullptr; pl->cap = 0;
        if (cudaMalloc(&pl->partials, (size_t)2 * nblk * sizeof(double)) != cudaSuccess) { err = "lq_descent: cudaMalloc failed"; return LQ_ERR_NOMEM; }
        pl->cap = (size_t)2 * nblk;
    }
    if (!pl->counter && cudaMalloc(&pl->counter, sizeof(unsigned int)) != cudaSuccess) { err = "lq_descent: cudaMalloc failed"; return LQ_ERR_NOMEM; }
    cudaError_t e = cudaMemsetAsync(pl->counter, 0, sizeof(unsigned int), st);
    if (e != cudaSuccess) { err = cudaGetErrorString(e); return LQ_ERR_CUDA; }

    DescArgs a;
    a.g = g; a.ph = ph; a.f = f; a.eta = eta; a.mu = nest ? mu : 0.0; a.force_tol = force_tol;
    a.list = nullptr; a.n = 0; a.sc = dsc; a.partials = pl->partials; a.extra = nullptr; a.n_extra = 0;
    a.counter = pl->counter; a.finish = 1;
    const long chunk = force_tol > 0.0 ? 100 : (1L << 30);
    long done = 0;
    while (done < max_steps) {
        const long n = (max_steps - done) < chunk ? (max_steps - done) : chunk;
        for (long i = 0; i < n; ++i) {
            const long k = done + i;
            const int in = (int)(k % nbuf), out = (int)((k + 1) % nbuf), prev = k == 0 ? in : (int)((k - 1) % nbuf);
            a.q = buf[in]; a.qp = buf[prev]; a.qo = buf[out];
            if (three) {
                if (nest) k_descent<true, true><<<nblk, DB, 0, st>>>(a);
                else k_descent<true, false><<<nblk, DB, 0, st>>>(a);
            } else {
                if (nest) k_descent<false, true><<<nblk, DB, 0, st>>>(a);
                else k_descent<false, false><<<nblk, DB, 0, st>>>(a);
            }
            e = cudaGetLastError();
            if (e != cudaSuccess) { err = std::string("lq_descent launch: ") + cudaGetErrorString(e); return LQ_ERR_CUDA; }
        }
        done += n;
        *launches += n;
        if (force_tol > 0.0) {
            e = cudaMemcpyAsync(h, dsc, sizeof(*h), cudaMemcpyDeviceToHost, st);
            if (e == cudaSuccess) e = cudaStreamSynchronize(st);
            if (e != cudaSuccess) { err = std::string("lq_descent: ") + cudaGetErrorString(e); return LQ_ERR_CUDA; }
            if (h->converged) break;
        }
    }
    e = cudaMemcpyAsync(h, dsc, sizeof(*h), cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) { err = std::string("lq_descent: ") + cudaGetErrorString(e); return LQ_ERR_CUDA; }
    *final = (int)(h->step % nbuf);
    return LQ_OK;
}

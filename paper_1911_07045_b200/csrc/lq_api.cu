// lq_api.cu -- the C ABI of liblq.so (include/lq.h): argument checking, device buffers,
// host<->device marshalling and the FIRE driver loop.  No arithmetic of the method runs on
// the host: every step of the path is a kernel in lq_kernels.cu / lq_sweep.cu.
#include "lq_ctx.cuh"

#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>
#include <string>

thread_local std::string g_noctx_err;

namespace {

}  // namespace

cudaError_t lq_copy_box(const LqGeom &g, const void *padded_c, const void *user, size_t elem, int ncomp, bool to_padded,
                        cudaStream_t st, int pz0, int nz, int user_z0, int user_nz) {
    void *padded = const_cast<void *>(padded_c);
    if (nz < 0) nz = g.Lz;
    if (user_nz < 0) user_nz = nz;
    for (int c = 0; c < ncomp; ++c) {
        cudaMemcpy3DParms p;
        memset(&p, 0, sizeof(p));
        cudaPitchedPtr up = make_cudaPitchedPtr((char *)user + (size_t)c * g.Lx * g.Ly * (size_t)user_nz * elem, g.Lx * elem,
                                                g.Lx * elem, g.Ly);
        cudaPitchedPtr pp = make_cudaPitchedPtr((char *)padded + (size_t)c * g.NP * elem, g.Px * elem, g.Px * elem, g.Py);
        cudaPos ppos = make_cudaPos(LQ_XO * elem, LQ_GH, pz0), upos = make_cudaPos(0, 0, user_z0);
        if (to_padded) { p.srcPtr = up; p.srcPos = upos; p.dstPtr = pp; p.dstPos = ppos; }
        else           { p.srcPtr = pp; p.srcPos = ppos; p.dstPtr = up; p.dstPos = upos; }
        p.extent = make_cudaExtent(g.Lx * elem, g.Ly, nz);
        p.kind = cudaMemcpyDefault;
        cudaError_t e = cudaMemcpy3DAsync(&p, st);
        if (e != cudaSuccess) return e;
    }
    return cudaSuccess;
}

int lq_ensure_field(lq_ctx *c, double **p) {
    if (*p) return LQ_OK;
    LQ_CUDA(c, cudaMalloc(p, (size_t)5 * c->g.NP * sizeof(double)));
    LQ_CUDA(c, cudaMemsetAsync(*p, 0, (size_t)5 * c->g.NP * sizeof(double), c->stream));
    return LQ_OK;
}

namespace {

int ensure_partials(lq_ctx *c, size_t n) {
    if (c->partials_len >= n) return LQ_OK;
    if (c->partials) cudaFree(c->partials);
    c->partials = nullptr; c->partials_len = 0;
    LQ_CUDA(c, cudaMalloc(&c->partials, n * sizeof(double)));
    c->partials_len = n;
    return LQ_OK;
}

}  // namespace

extern "C" {

const char *lq_version(void) { return "lq 0.1 sm_100a"; }

const char *lq_last_error(lq_ctx *ctx) { return ctx ? ctx->err.c_str() : g_noctx_err.c_str(); }

int lq_create(int Lx, int Ly, int Lz, double A, double B, double C, double L1, double L2, double L3, lq_ctx **out) {
    if (!out) return fail(nullptr, LQ_ERR_ARG, "lq_create: out is NULL");
    *out = nullptr;
    if (Lx < 4 || Ly < 4 || Lz < 4) return fail(nullptr, LQ_ERR_ARG, "lq_create: every lattice dimension must be >= 4");
    if (!(C > 0.0) || !(B * B - 24.0 * A * C >= 0.0))
        return fail(nullptr, LQ_ERR_ARG, "lq_create: need C > 0 and B^2 - 24AC >= 0 (Eq. 7 has no nematic minimum)");
    if (!std::isfinite(A) || !std::isfinite(B) || !std::isfinite(L1) || !std::isfinite(L2) || !std::isfinite(L3))
        return fail(nullptr, LQ_ERR_ARG, "lq_create: non-finite constant");
    int ndev = 0;
    cudaError_t e = cudaGetDeviceCount(&ndev);
    if (e != cudaSuccess || ndev == 0)
        return fail(nullptr, LQ_ERR_CUDA, std::string("lq_create: no CUDA device (there is no CPU fallback): ") +
                                              cudaGetErrorString(e));
    int dev = 0;
    cudaGetDevice(&dev);
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, dev) != cudaSuccess || prop.major != 10)
        return fail(nullptr, LQ_ERR_CUDA, "lq_create: device is not sm_100 (this library is built for sm_100a only)");

    lq_ctx *c = new (std::nothrow) lq_ctx();
    if (!c) return fail(nullptr, LQ_ERR_NOMEM, "lq_create: out of host memory");
    c->device = dev;
    LqGeom &g = c->g;
    g.Lx = Lx; g.Ly = Ly; g.Lz = Lz;
    g.Px = ((LQ_XO + Lx + LQ_GH + 15) / 16) * 16;
    g.Py = Ly + 2 * LQ_GH; g.Pz = Lz + 2 * LQ_GH;
    g.sy = g.Px; g.sz = (long long)g.Px * g.Py;
    g.NP = g.sz * g.Pz; g.N = (long long)Lx * Ly * Lz;
    g.gwx = (Lx % 4 == 0 && Lx >= 8 && g.Px - LQ_XO - Lx >= 4) ? 4 : LQ_GH;
    if (g.NP > 2147483647LL) { delete c; return fail(nullptr, LQ_ERR_ARG, "lq_create: lattice too large (padded sites > 2^31-1)"); }
    c->ph = LqPhys{A, B, C, L1, L2, L3, (-B + sqrt(B * B - 24.0 * A * C)) / (6.0 * C)};
    int rc = LQ_OK;
    do {
        if ((rc = lq_ensure_field(c, &c->q[0])) != LQ_OK) break;
        if (cudaMalloc(&c->dscal3, 3 * sizeof(double)) != cudaSuccess ||
            cudaMalloc(&c->dsc, 2 * sizeof(LqFireScalars)) != cudaSuccess ||
            cudaMalloc(&c->dcounts, 3 * sizeof(unsigned long long)) != cudaSuccess ||
            cudaMalloc(&c->dbad, 2 * sizeof(int)) != cudaSuccess) {
            rc = fail(nullptr, LQ_ERR_NOMEM, "lq_create: cudaMalloc failed");
            break;
        }
        if (cudaEventCreate(&c->ev0) != cudaSuccess || cudaEventCreate(&c->ev1) != cudaSuccess) {
            rc = fail(nullptr, LQ_ERR_CUDA, "lq_create: cudaEventCreate failed");
            break;
        }
    } while (0);
    if (rc != LQ_OK) { std::string m = c->err.empty() ? g_noctx_err : c->err; lq_destroy(c); return fail(nullptr, rc, m); }
    *out = c;
    return LQ_OK;
}

void lq_destroy(lq_ctx *c) {
    if (!c) return;
    DeviceGuard dg(c);
    if (c->ev0) cudaEventDestroy(c->ev0);
    if (c->ev1) cudaEventDestroy(c->ev1);
    cudaFree(c->res_bond);
    cudaFree(c->scratch); cudaFree(c->dtot); cudaFree(c->dsegs); cudaFree(c->dscptr);
    for (int i = 0; i < 2; ++i) { cudaFree(c->q[i]); cudaFree(c->v[i]); cudaFree(c->F[i]); }
    cudaFree(c->maskp); cudaFree(c->flags); cudaFree(c->kind); cudaFree(c->W); cudaFree(c->axis);
    cudaFree(c->partials); cudaFree(c->dscal3); cudaFree(c->dsc); cudaFree(c->dcounts); cudaFree(c->dbad);
    lq_sweep_destroy(c->sweep);
    lq_descent_destroy(c->descent);
    delete c;
}

int lq_set_stream(lq_ctx *c, void *s) {
    if (!c) return LQ_ERR_ARG;
    DeviceGuard dg(c);
    c->stream = (cudaStream_t)s;
    return LQ_OK;
}

int lq_set_sites(lq_ctx *c, const uint8_t *mask, const uint8_t *anch_kind, const double *W, const double *axis,
                 int where) {
    if (!c) return LQ_ERR_ARG;
    DeviceGuard dg(c);
    if (bad_where(where)) return fail(c, LQ_ERR_ARG, "lq_set_sites: bad `where`");
    if (c->g.zopen && mask) return fail(c, LQ_ERR_STATE, "lq_set_sites: sub-domain contexts take lq_set_sites_ext (arrays with a 3-plane margin)");
    if (anch_kind && (!W || !axis)) return fail(c, LQ_ERR_ARG, "lq_set_sites: anch_kind given without W / axis");
    const LqGeom &g = c->g;
    cudaStream_t st = c->stream;
    if (!mask) {
        lq_sweep_invalidate(c->sweep);
        lq_descent_invalidate(c->descent);
        c->res_bond_dirty = true;
        c->flags_active = false; c->anch_active = false;
        c->n_class[0] = (unsigned long long)g.N; c->n_class[1] = c->n_class[2] = 0;
        return LQ_OK;
    }
    // 1. stage the inputs and validate them; the context's geometry state changes only after both checks passed
    //    (the staging arrays themselves are scratch until then: on a bad input the sites are reset to "all bulk")
    if (!c->maskp) LQ_CUDA(c, cudaMalloc(&c->maskp, (size_t)g.NP));
    if (!c->flags) LQ_CUDA(c, cudaMalloc(&c->flags, (size_t)g.NP));
    LQ_CUDA(c, cudaMemsetAsync(c->maskp, 0, (size_t)g.NP, st));
    LQ_CUDA(c, lq_copy_box(g, c->maskp, mask, 1, 1, true, st));
    LQ_CUDA(c, cudaMemsetAsync(c->dbad, 0, 2 * sizeof(int), st));
    lq_launch_check_u8_max(g, c->maskp, 1, c->dbad, st);
    if (anch_kind) {
        if (!c->kind) LQ_CUDA(c, cudaMalloc(&c->kind, (size_t)g.NP));
        if (!c->W) LQ_CUDA(c, cudaMalloc(&c->W, (size_t)g.NP * sizeof(double)));
        if (!c->axis) LQ_CUDA(c, cudaMalloc(&c->axis, (size_t)3 * g.NP * sizeof(double)));
        LQ_CUDA(c, cudaMemsetAsync(c->kind, 0, (size_t)g.NP, st));
        LQ_CUDA(c, lq_copy_box(g, c->kind, anch_kind, 1, 1, true, st));
        lq_launch_check_u8_max(g, c->kind, 2, c->dbad + 1, st);
    }
    int bad[2] = {0, 0};
    LQ_CUDA(c, cudaMemcpyAsync(bad, c->dbad, 2 * sizeof(int), cudaMemcpyDeviceToHost, st));
    LQ_CUDA(c, cudaStreamSynchronize(st));
    lq_sweep_invalidate(c->sweep);
    lq_descent_invalidate(c->descent);
    c->res_bond_dirty = true;
    if (bad[0] || (anch_kind && bad[1])) {
        c->flags_active = false; c->anch_active = false;
        c->n_class[0] = (unsigned long long)g.N; c->n_class[1] = c->n_class[2] = 0;
        return fail(c, LQ_ERR_ARG, bad[0] ? "lq_set_sites: mask value > 1 (sites reset to all bulk)"
                                          : "lq_set_sites: anch_kind value > 2 (sites reset to all bulk)");
    }
    // 2. classify
    LQ_CUDA(c, cudaMemsetAsync(c->flags, 0xFC, (size_t)g.NP, st));
    lq_launch_fill_ghosts_u8(g, c->maskp, st);
    lq_launch_classify(g, c->maskp, c->flags, st);
    lq_launch_fill_ghosts_u8(g, c->flags, st);
    LQ_CUDA(c, cudaMemsetAsync(c->dcounts, 0, 3 * sizeof(unsigned long long), st));
    lq_launch_count_classes(g, c->flags, c->dcounts, st);
    if (anch_kind) {
        LQ_CUDA(c, cudaMemsetAsync(c->W, 0, (size_t)g.NP * sizeof(double), st));
        LQ_CUDA(c, cudaMemsetAsync(c->axis, 0, (size_t)3 * g.NP * sizeof(double), st));
        LQ_CUDA(c, lq_copy_box(g, c->W, W, sizeof(double), 1, true, st));
        LQ_CUDA(c, lq_copy_box(g, c->axis, axis, sizeof(double), 3, true, st));
        lq_launch_fill_ghosts_u8(g, c->kind, st);     // the recompute sweep evaluates anchoring on halo sites
        lq_launch_fill_ghosts_f64(g, c->W, 1, st);
        lq_launch_fill_ghosts_f64(g, c->axis, 3, st);
    }
    LQ_CUDA(c, cudaMemcpyAsync(c->n_class, c->dcounts, 3 * sizeof(unsigned long long), cudaMemcpyDeviceToHost, st));
    LQ_CUDA(c, cudaStreamSynchronize(st));
    LQ_CUDA(c, cudaGetLastError());
    c->flags_active = c->n_class[2] > 0;
    c->anch_active = anch_kind != nullptr && c->n_class[1] > 0;
    return LQ_OK;
}

int lq_get_flags(lq_ctx *c, uint8_t *flags, int where) {
    if (!c) return LQ_ERR_ARG;
    DeviceGuard dg(c);
    if (!flags || bad_where(where)) return fail(c, LQ_ERR_ARG, "lq_get_flags: bad argument");
    if (!c->flags_active) {
        if (where == LQ_HOST) memset(flags, 0xFC, (size_t)c->g.N);
        else LQ_CUDA(c, cudaMemsetAsync(flags, 0xFC, (size_t)c->g.N, c->stream));
    } else {
        LQ_CUDA(c, lq_copy_box(c->g, c->flags, flags, 1, 1, false, c->stream));
    }
    LQ_CUDA(c, cudaStreamSynchronize(c->stream));
    return LQ_OK;
}

int lq_set_Q(lq_ctx *c, const double *q, int where) {
    if (!c) return LQ_ERR_ARG;
    DeviceGuard dg(c);
    if (!q || bad_where(where)) return fail(c, LQ_ERR_ARG, "lq_set_Q: bad argument");
    LQ_CUDA(c, lq_copy_box(c->g, c->q[c->cur], q, sizeof(double), 5, true, c->stream));
    lq_launch_fill_ghosts_f64(c->g, c->q[c->cur], 5, c->stream);
    LQ_CUDA(c, cudaStreamSynchronize(c->stream));
    LQ_CUDA(c, cudaGetLastError());
    c->has_Q = true;
    c->v_valid = false;        // velocities read as zero until the next lq_fire_minimize (no 40 B/site memset here)
    return LQ_OK;
}

int lq_get_Q(lq_ctx *c, double *q, int where) {
    if (!c) return LQ_ERR_ARG;
    DeviceGuard dg(c);
    if (!q || bad_where(where)) return fail(c, LQ_ERR_ARG, "lq_get_Q: bad argument");
    if (!c->has_Q) return fail(c, LQ_ERR_STATE, "lq_get_Q: no Q has been set");
    LQ_CUDA(c, lq_copy_box(c->g, c->q[c->cur], q, sizeof(double), 5, false, c->stream));
    LQ_CUDA(c, cudaStreamSynchronize(c->stream));
    return LQ_OK;
}

int lq_get_velocity(lq_ctx *c, double *v, int where) {
    if (!c) return LQ_ERR_ARG;
    DeviceGuard dg(c);
    if (!v || bad_where(where)) return fail(c, LQ_ERR_ARG, "lq_get_velocity: bad argument");
    if (!c->has_Q) return fail(c, LQ_ERR_STATE, "lq_get_velocity: no Q has been set");
    int rc = lq_ensure_field(c, &c->v[c->cur]);
    if (rc != LQ_OK) return rc;
    if (!c->v_valid) {
        LQ_CUDA(c, cudaMemsetAsync(c->v[c->cur], 0, (size_t)5 * c->g.NP * sizeof(double), c->stream));
        c->v_valid = true; c->v_mix_a = 1.0; c->v_mix_b = 0.0;
    }
    const double *src = c->v[c->cur];
    if (c->v_mix_a != 1.0 || c->v_mix_b != 0.0) {
        // the last step's rescale v <- (1-alpha) v + alpha |v| F/|F| (or v <- 0) is still pending: apply it to a copy
        if ((rc = lq_ensure_field(c, &c->F[c->cur])) != LQ_OK) return rc;
        lq_launch_forces(c->g, c->ph, fields_of(c), c->q[c->cur], c->F[c->cur], c->stream);
        lq_launch_axpby((long long)5 * c->g.NP, c->v_mix_a, c->v[c->cur], c->v_mix_b, c->F[c->cur], c->F[c->cur], c->stream);
        src = c->F[c->cur];
    }
    LQ_CUDA(c, lq_copy_box(c->g, src, v, sizeof(double), 5, false, c->stream));
    LQ_CUDA(c, cudaStreamSynchronize(c->stream));
    return LQ_OK;
}

int lq_energy_terms(lq_ctx *c, double *terms) {
    if (!c) return LQ_ERR_ARG;
    DeviceGuard dg(c);
    if (!terms) return fail(c, LQ_ERR_ARG, "lq_energy_terms: terms is NULL");
    if (!c->has_Q) return fail(c, LQ_ERR_STATE, "lq_energy: no Q has been set");
    int rc = ensure_partials(c, (size_t)3 * lq_energy_num_blocks(c->g));
    if (rc != LQ_OK) return rc;
    lq_launch_energy(c->g, c->ph, fields_of(c), c->q[c->cur], c->partials, c->dscal3, c->stream);
    LQ_CUDA(c, cudaMemcpyAsync(terms, c->dscal3, 3 * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    LQ_CUDA(c, cudaStreamSynchronize(c->stream));
    LQ_CUDA(c, cudaGetLastError());
    return LQ_OK;
}

int lq_energy(lq_ctx *c, double *E) {
    if (!c) return LQ_ERR_ARG;
    DeviceGuard dg(c);
    if (!E) return fail(c, LQ_ERR_ARG, "lq_energy: E is NULL");
    double t[3];
    int rc = lq_energy_terms(c, t);
    if (rc != LQ_OK) return rc;
    *E = t[0] + t[1] + t[2];
    return LQ_OK;
}

int lq_forces(lq_ctx *c, double *F, int where) {
    if (!c) return LQ_ERR_ARG;
    DeviceGuard dg(c);
    if (!F || bad_where(where)) return fail(c, LQ_ERR_ARG, "lq_forces: bad argument");
    if (!c->has_Q) return fail(c, LQ_ERR_STATE, "lq_forces: no Q has been set");
    int rc = lq_ensure_field(c, &c->F[c->cur]);
    if (rc != LQ_OK) return rc;
    lq_launch_forces(c->g, c->ph, fields_of(c), c->q[c->cur], c->F[c->cur], c->stream);
    LQ_CUDA(c, lq_copy_box(c->g, c->F[c->cur], F, sizeof(double), 5, false, c->stream));
    LQ_CUDA(c, cudaStreamSynchronize(c->stream));
    LQ_CUDA(c, cudaGetLastError());
    return LQ_OK;
}

int lq_get_S0(lq_ctx *c, double *S0) {
    if (!c || !S0) return LQ_ERR_ARG;
    *S0 = c->ph.S0;
    return LQ_OK;
}

int lq_set_option(lq_ctx *c, const char *key, double value) {
    if (!c || !key) return LQ_ERR_ARG;
    DeviceGuard dg(c);
    if (!strcmp(key, "fire_path")) {
        if (value != 0.0 && value != 1.0 && value != 2.0) return fail(c, LQ_ERR_ARG, "fire_path must be 0, 1 or 2");
        c->fire_path = (int)value;
        return LQ_OK;
    }
    if (!strcmp(key, "resident")) {
        if (value != 0.0 && value != 1.0) return fail(c, LQ_ERR_ARG, "resident must be 0 or 1");
        c->resident = (int)value;
        return LQ_OK;
    }
    if (!strcmp(key, "rc_chunks")) {
        if (!(value >= 0.0 && value <= 4096.0)) return fail(c, LQ_ERR_ARG, "rc_chunks must be in [0, 4096]");
        c->rc_chunks = (int)value;
        return LQ_OK;
    }
    return fail(c, LQ_ERR_ARG, std::string("lq_set_option: unknown key ") + key);
}

int lq_get_info(lq_ctx *c, const char *key, double *value) {
    if (!c || !key || !value) return LQ_ERR_ARG;
    const double nsim = (double)(c->flags_active ? c->n_class[0] + c->n_class[1] : (unsigned long long)c->g.N);
    if (!strcmp(key, "n_simulated")) { *value = nsim; return LQ_OK; }
    if (!strcmp(key, "n_boundary")) { *value = c->flags_active ? (double)c->n_class[1] : 0.0; return LQ_OK; }
    if (!strcmp(key, "n_object")) { *value = c->flags_active ? (double)c->n_class[2] : 0.0; return LQ_OK; }
    if (!strcmp(key, "has_fixup")) {      // FIRE step = sweep + fix-up launch (stored force on a lattice with objects)
        *value = ((lq_three(c->ph) || c->fire_path == 2) && c->flags_active) ? 1.0 : 0.0;
        return LQ_OK;
    }
    if (!strcmp(key, "stored_force")) { *value = (lq_three(c->ph) || c->fire_path == 2) ? 1.0 : 0.0; return LQ_OK; }
    if (!strcmp(key, "fire_sweeps_total")) {     // step-wise FIRE of a sub-domain: rounds a full run takes (lq.h)
        if (!c->fire_open) return fail(c, LQ_ERR_STATE, "lq_get_info: fire_sweeps_total is defined between lq_fire_begin and lq_fire_end");
        const bool extra = lq_three(c->ph) || c->fire_path == 2 || c->fire_fc.euler;
        const long long m = c->fire_fc.max_steps;
        *value = (double)(extra ? m + 1 : (m > 0 ? m : 1));
        return LQ_OK;
    }
    if (!strcmp(key, "fp64_fma_tflops")) {       // measured now: the fp64 ALU roof of this device (a few ms of FMAs)
        DeviceGuard dg(c);
        const double t = lq_measure_fp64_fma(c->device, c->stream);
        if (t < 0.0) return fail(c, LQ_ERR_CUDA, "lq_get_info: the fp64 FMA microbenchmark failed");
        *value = t;
        return LQ_OK;
    }
    if (!strcmp(key, "sweep_bytes_per_site")) {
        // fused sweep: read + write q, v (and F when it is stored), 5 fp64 each, + the flag byte where objects exist
        const bool three = lq_three(c->ph);
        const double fields = (three || c->fire_path == 2) ? 6.0 : 4.0;
        *value = c->fire_path == 1 ? 0.0 : fields * 40.0 + (c->flags_active ? 1.0 : 0.0);
        return LQ_OK;
    }
    return fail(c, LQ_ERR_ARG, std::string("lq_get_info: unknown key ") + key);
}

int lq_fire_minimize(lq_ctx *c, long max_steps, double force_tol, const lq_fire_params *fp, lq_fire_report *out) {
    if (!c) return LQ_ERR_ARG;
    DeviceGuard dg(c);
    if (!fp || !out) return fail(c, LQ_ERR_ARG, "lq_fire_minimize: NULL params / report");
    if (!c->has_Q) return fail(c, LQ_ERR_STATE, "lq_fire_minimize: no Q has been set");
    if (c->g.zopen) return fail(c, LQ_ERR_STATE, "lq_fire_minimize: sub-domain contexts run lq_slabs_fire_minimize or lq_fire_begin / step / end");
    if (!(fp->dt0 > 0.0) || !(fp->dtmax >= fp->dt0) || !(fp->alpha0 >= 0.0 && fp->alpha0 <= 1.0) ||
        !(fp->finc >= 1.0) || !(fp->fdec > 0.0 && fp->fdec <= 1.0) || !(fp->falpha > 0.0 && fp->falpha <= 1.0) ||
        fp->Nmin < 0 || (fp->integrator != 0 && fp->integrator != 1) || max_steps < 0 || !(force_tol >= 0.0))
        return fail(c, LQ_ERR_ARG, "lq_fire_minimize: bad FIRE parameter");
    memset(out, 0, sizeof(*out));
    const LqGeom &g = c->g;
    cudaStream_t st = c->stream;
    int rc;
    const bool euler = fp->integrator == 1;
    const bool fused = c->fire_path != 1;
    const bool three = lq_three(c->ph);
    const bool stored_F = three || c->fire_path == 2;   // recompute-F sweep: one-constant only
    if ((rc = lq_ensure_field(c, &c->v[c->cur])) != LQ_OK) return rc;
    if ((!fused || stored_F) && (rc = lq_ensure_field(c, &c->F[c->cur])) != LQ_OK) return rc;
    if (fused) {
        if ((rc = lq_ensure_field(c, &c->q[c->cur ^ 1])) != LQ_OK) return rc;
        if ((rc = lq_ensure_field(c, &c->v[c->cur ^ 1])) != LQ_OK) return rc;
        if (stored_F && (rc = lq_ensure_field(c, &c->F[c->cur ^ 1])) != LQ_OK) return rc;
    }

    LqFireConsts fc{fp->dt0, fp->dtmax, fp->alpha0, fp->finc, fp->fdec, fp->falpha, force_tol, fp->Nmin, (long long)max_steps,
                    euler ? 1 : 0};
    LqFireScalars h;
    memset(&h, 0, sizeof(h));
    const LqFields f = fields_of(c);
    long launches = 0, sweeps = 0;
    LQ_CUDA(c, cudaEventRecord(c->ev0, st));

    bool done_resident = false;
    int rdims[6];
    int nsm = 148;
    cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, c->device);
    if (fused && !stored_F && !euler && c->resident && lq_resident_plan(g, nsm, rdims)) {
        // small lattice: the whole call is ONE cooperative launch with the state resident on chip (lq_resident.cu)
        const int ncta = rdims[0] * rdims[1] * rdims[2];
        if ((rc = ensure_partials(c, (size_t)10 * ncta)) != LQ_OK) return rc;
        for (int i = 0; i < 2; ++i)
            if ((rc = lq_ensure_field(c, &c->F[i])) != LQ_OK) return rc;
        if (f.flags && c->res_bond_dirty) {
            if (!c->res_bond) LQ_CUDA(c, cudaMalloc(&c->res_bond, (size_t)g.NP * sizeof(uint32_t)));
            LQ_CUDA(c, cudaMemsetAsync(c->res_bond, 0, (size_t)g.NP * sizeof(uint32_t), st));
            lq_launch_bond_map(g, f.flags, f.kind, c->res_bond, st);
            c->res_bond_dirty = false;
            launches += 1;
        }
        h.dt = fp->dt0; h.alpha = fp->alpha0;
        LQ_CUDA(c, cudaMemcpyAsync(&c->dsc[0], &h, sizeof(h), cudaMemcpyHostToDevice, st));
        cudaError_t e = lq_launch_fire_resident(g, c->ph, f, c->q, c->v, c->F, c->cur, f.flags ? c->res_bond : nullptr,
                                                c->dsc, fc, c->partials, rdims, st);
        if (e == cudaSuccess) {
            LQ_CUDA(c, cudaMemcpyAsync(&h, &c->dsc[0], sizeof(h), cudaMemcpyDeviceToHost, st));
            LQ_CUDA(c, cudaStreamSynchronize(st));
            // the final state sits in the buffer the last step wrote; the kernel writes interiors only: refresh the
            // periodic ghost shells of q and v for whatever runs next
            c->cur = (int)((c->cur + h.step) & 1);
            lq_launch_fill_ghosts_f64(g, c->q[c->cur], 5, st);
            lq_launch_fill_ghosts_f64(g, c->v[c->cur], 5, st);
            launches += 3; sweeps += 1;
            done_resident = true;
        } else if (e != cudaErrorCooperativeLaunchTooLarge) {
            return fail(c, LQ_ERR_CUDA, std::string("lq_fire_minimize (resident kernel): ") + cudaGetErrorString(e));
        } else {
            cudaGetLastError();          // not co-resident on this device: the streaming sweeps take over
            memset(&h, 0, sizeof(h));
        }
    }
    if (done_resident) {
    } else if (fused) {
        // Algorithm 1's initialisation (v = 0, dt0, alpha0, force of the initial state and the stop test on it) is
        // part of the first sweep: mix_a = mix_b = 0 makes it ignore whatever the velocity buffer holds, the
        // recompute sweep reduces max|F(q_0)| in its first phase, the stored-force path starts with one sweep whose
        // step coefficients are all 0 (init), the Euler variant with its own [no drift | force | kick] sweep.
        h.dt = fp->dt0; h.alpha = fp->alpha0; h.mix_a = 0.0; h.mix_b = 0.0; h.dt_prev = 0.0;
        h.init = (stored_F && !euler) ? 1 : 0;
        LQ_CUDA(c, cudaMemcpyAsync(&c->dsc[0], &h, sizeof(h), cudaMemcpyHostToDevice, st));
        // build the plan first (tensor maps, the host-side search of the chunk table, set-up kernels: all on the first
        // call only) and restart the clock, so that report.gpu_ms is the device time of the sweeps alone
        if ((rc = lq_sweep_prepare(&c->sweep, stored_F, g, c->ph, f, c->q, c->v, c->F, st, &launches, c->err, c->rc_chunks)) != LQ_OK)
            return rc;
        LQ_CUDA(c, cudaEventRecord(c->ev0, st));
        rc = lq_sweep_run(&c->sweep, stored_F, g, c->ph, f, c->q, c->v, c->F, &c->cur, c->dsc, fc, max_steps, st, &launches,
                          &sweeps, &h, c->err, c->rc_chunks);
        if (rc != LQ_OK) return rc;
    } else {
        // unfused cross-check path (fire_path = 1): generic one-thread-per-site kernels, 4 launches per step
        const int nb1 = lq_fire1_num_blocks(g);
        if ((rc = ensure_partials(c, (size_t)4 * nb1)) != LQ_OK) return rc;
        h.dt = euler ? fp->dt0 : 0.0; h.alpha = fp->alpha0; h.mix_a = 1.0; h.mix_b = 0.0;
        LQ_CUDA(c, cudaMemcpyAsync(&c->dsc[0], &h, sizeof(h), cudaMemcpyHostToDevice, st));
        LQ_CUDA(c, cudaMemsetAsync(c->v[c->cur], 0, (size_t)5 * g.NP * sizeof(double), st));
        // step 0: F = force(q), convergence test on the initial state (dt = 0: no kick)
        // (Euler variant: the same launch is the first step's full kick v += dt0 F and its reductions)
        const long long emax = euler ? (long long)max_steps : -1;
        lq_launch_fire1_force(g, c->ph, f, c->q[c->cur], c->v[c->cur], c->F[c->cur], &c->dsc[0], c->partials, st, emax);
        lq_launch_fire_update(c->partials, nb1, &c->dsc[0], fc, euler ? 2 : 1, st);
        launches += 2;
        long done = 0;
        const long chunk = force_tol > 0.0 ? 64 : 1024;
        while (done < max_steps) {
            const long n = (max_steps - done) < chunk ? (max_steps - done) : chunk;
            for (long i = 0; i < n; ++i) {
                lq_launch_fire1_drift(g, f, c->q[c->cur], c->v[c->cur], c->F[c->cur], &c->dsc[0], st, euler ? 1 : 0);
                lq_launch_fill_ghosts_f64(g, c->q[c->cur], 5, st);
                lq_launch_fire1_force(g, c->ph, f, c->q[c->cur], c->v[c->cur], c->F[c->cur], &c->dsc[0], c->partials, st, emax);
                lq_launch_fire_update(c->partials, nb1, &c->dsc[0], fc, euler ? 2 : 0, st);
            }
            launches += 4 * n;
            done += n;
            if (force_tol > 0.0) {
                LQ_CUDA(c, cudaMemcpyAsync(&h, &c->dsc[0], sizeof(h), cudaMemcpyDeviceToHost, st));
                LQ_CUDA(c, cudaStreamSynchronize(st));
                if (h.converged) break;
            }
        }
        LQ_CUDA(c, cudaMemcpyAsync(&h, &c->dsc[0], sizeof(h), cudaMemcpyDeviceToHost, st));
    }
    LQ_CUDA(c, cudaEventRecord(c->ev1, st));
    LQ_CUDA(c, cudaStreamSynchronize(st));
    LQ_CUDA(c, cudaGetLastError());
    float ms = 0.f;
    cudaEventElapsedTime(&ms, c->ev0, c->ev1);
    // velocities: the buffer holds the last step's v only if a step ran (a stop on the initial state leaves v = 0)
    c->v_valid = h.step > 0 || !fused;
    const bool pending = !h.converged && h.step > 0 && !(euler && h.step >= (long long)max_steps);
    c->v_mix_a = pending ? h.mix_a : 1.0;
    c->v_mix_b = pending ? h.mix_b : 0.0;

    const double nsim = (double)(c->flags_active ? c->n_class[0] + c->n_class[1] : (unsigned long long)g.N);
    out->steps = (long)h.step; out->converged = h.converged;
    out->Fmax = h.Fmax; out->Frms = nsim > 0 ? sqrt(h.FF / nsim) : 0.0;
    out->P = h.P; out->dt = h.dt; out->alpha = h.alpha;
    out->launches = launches; out->sweep_launches = sweeps; out->gpu_ms = ms;
    if (fp->report_energy) {
        rc = lq_energy(c, &out->energy);
        if (rc != LQ_OK) return rc;
    }
    return LQ_OK;
}


int lq_analyze(lq_ctx *c, double thr, double *S, double *dir, uint8_t *defect, long *n_defect, int where) {
    if (!c) return LQ_ERR_ARG;
    DeviceGuard dg(c);
    if (bad_where(where)) return fail(c, LQ_ERR_ARG, "lq_analyze: bad `where`");
    if (!c->has_Q) return fail(c, LQ_ERR_STATE, "lq_analyze: call lq_set_Q first");
    const LqGeom &g = c->g;
    cudaStream_t st = c->stream;
    const size_t N = (size_t)g.N;
    double *dS = S, *dD = dir;
    uint8_t *dF = defect;
    if (where == LQ_HOST) {                     // stage through device scratch kept in the context
        const size_t need = (S ? N * sizeof(double) : 0) + (dir ? 3 * N * sizeof(double) : 0) + (defect ? N : 0);
        if (need > c->scratch_len) {
            cudaFree(c->scratch);
            c->scratch = nullptr; c->scratch_len = 0;
            LQ_CUDA(c, cudaMalloc(&c->scratch, need));
            c->scratch_len = need;
        }
        char *sp = (char *)c->scratch;
        if (S) { dS = (double *)sp; sp += N * sizeof(double); }
        if (dir) { dD = (double *)sp; sp += 3 * N * sizeof(double); }
        if (defect) dF = (uint8_t *)sp;
    }
    LQ_CUDA(c, cudaMemsetAsync(c->dcounts, 0, sizeof(unsigned long long), st));
    lq_launch_analyze(g, c->q[c->cur], c->flags_active ? c->flags : nullptr, thr, dS, dD, dF, c->dcounts, st);
    LQ_CUDA(c, cudaGetLastError());
    unsigned long long cnt = 0;
    LQ_CUDA(c, cudaMemcpyAsync(&cnt, c->dcounts, sizeof(cnt), cudaMemcpyDeviceToHost, st));
    if (where == LQ_HOST) {
        if (S) LQ_CUDA(c, cudaMemcpyAsync(S, dS, N * sizeof(double), cudaMemcpyDeviceToHost, st));
        if (dir) LQ_CUDA(c, cudaMemcpyAsync(dir, dD, 3 * N * sizeof(double), cudaMemcpyDeviceToHost, st));
        if (defect) LQ_CUDA(c, cudaMemcpyAsync(defect, dF, N, cudaMemcpyDeviceToHost, st));
    }
    LQ_CUDA(c, cudaStreamSynchronize(st));
    if (n_defect) *n_defect = (long)cnt;
    return LQ_OK;
}

int lq_set_chiral(lq_ctx *c, double L4) {
    if (!c) return LQ_ERR_ARG;
    DeviceGuard dg(c);
    if (!std::isfinite(L4)) return fail(c, LQ_ERR_ARG, "lq_set_chiral: non-finite L4");
    c->ph.L4 = L4;
    return LQ_OK;
}

int lq_set_cubic(lq_ctx *c, double L6) {
    if (!c) return LQ_ERR_ARG;
    DeviceGuard dg(c);
    if (!std::isfinite(L6)) return fail(c, LQ_ERR_ARG, "lq_set_cubic: non-finite L6");
    c->ph.L6 = L6;
    return LQ_OK;
}

int lq_set_field(lq_ctx *c, const double *H, double chi, const double *E, double eps) {
    if (!c) return LQ_ERR_ARG;
    DeviceGuard dg(c);
    double h[3] = {0.0, 0.0, 0.0}, e[3] = {0.0, 0.0, 0.0};
    for (int i = 0; i < 3; ++i) {
        if (H) h[i] = H[i];
        if (E) e[i] = E[i];
        if (!std::isfinite(h[i]) || !std::isfinite(e[i])) return fail(c, LQ_ERR_ARG, "lq_set_field: non-finite field");
    }
    if (!std::isfinite(chi) || !std::isfinite(eps)) return fail(c, LQ_ERR_ARG, "lq_set_field: non-finite coefficient");
    const int ia[6] = {0, 0, 0, 1, 1, 2}, ib[6] = {0, 1, 2, 1, 2, 2};      // (xx, xy, xz, yy, yz, zz)
    double *T = c->ph.T;
    for (int k = 0; k < 6; ++k) T[k] = (chi * h[ia[k]] * h[ib[k]] + eps * e[ia[k]] * e[ib[k]]) / 3.0;
    // F = -(Gxx - Gzz, 2 Gxy, 2 Gxz, Gyy - Gzz, 2 Gyz) with G_ab = -T_ab
    c->ph.Fx[0] = T[0] - T[5]; c->ph.Fx[1] = 2.0 * T[1]; c->ph.Fx[2] = 2.0 * T[2];
    c->ph.Fx[3] = T[3] - T[5]; c->ph.Fx[4] = 2.0 * T[4];
    return LQ_OK;
}

int lq_descent_minimize(lq_ctx *c, int method, long max_steps, double force_tol, const lq_descent_params *dp,
                        lq_fire_report *out) {
    if (!c) return LQ_ERR_ARG;
    DeviceGuard dg(c);
    if (!dp || !out) return fail(c, LQ_ERR_ARG, "lq_descent_minimize: NULL pointer");
    memset(out, 0, sizeof(*out));
    if (!c->has_Q) return fail(c, LQ_ERR_STATE, "lq_descent_minimize: call lq_set_Q first");
    if (c->g.zopen) return fail(c, LQ_ERR_STATE, "lq_descent_minimize: not available on sub-domain contexts");
    if ((method != LQ_MIN_GD && method != LQ_MIN_NESTEROV) || !(dp->eta > 0.0) || max_steps < 0 || !(force_tol >= 0.0) ||
        (method == LQ_MIN_NESTEROV && !(dp->mu >= 0.0 && dp->mu < 1.0)))
        return fail(c, LQ_ERR_ARG, "lq_descent_minimize: bad parameters");
    const LqGeom &g = c->g;
    cudaStream_t st = c->stream;
    int rc;
    const int nbuf = method == LQ_MIN_NESTEROV ? 3 : 2;
    if ((rc = lq_ensure_field(c, &c->q[c->cur ^ 1])) != LQ_OK) return rc;
    if (nbuf == 3 && (rc = lq_ensure_field(c, &c->v[0])) != LQ_OK) return rc;
    double *buf[3] = {c->q[c->cur], c->q[c->cur ^ 1], c->v[0]};
    LqFireScalars h;
    memset(&h, 0, sizeof(h));
    h.dt = dp->eta; h.alpha = dp->mu;
    LQ_CUDA(c, cudaMemcpyAsync(&c->dsc[0], &h, sizeof(h), cudaMemcpyHostToDevice, st));
    LQ_CUDA(c, cudaEventRecord(c->ev0, st));
    long launches = 0, sweeps = 0;
    int fin = 0;
    rc = lq_descent_run(&c->descent, method, c->fire_path == 1 ? 1 : 0, g, c->ph, fields_of(c), buf, nbuf, &fin, c->dsc,
                        dp->eta, dp->mu, force_tol, max_steps, st, &launches, &sweeps, &h, c->err);
    if (rc != LQ_OK) return rc;
    LQ_CUDA(c, cudaEventRecord(c->ev1, st));
    LQ_CUDA(c, cudaStreamSynchronize(st));
    float ms = 0.f;
    cudaEventElapsedTime(&ms, c->ev0, c->ev1);
    // make the buffer that holds the last iterate the live one
    if (fin == 1) c->cur ^= 1;
    else if (fin == 2) { double *t = c->q[c->cur]; c->q[c->cur] = c->v[0]; c->v[0] = t; }
    // these minimisers carry no velocity; the velocity storage may have served as their third buffer
    c->v_valid = false;
    const double nsim = (double)(c->flags_active ? c->n_class[0] + c->n_class[1] : (unsigned long long)g.N);
    out->steps = (long)h.step; out->converged = h.converged;
    out->Fmax = h.Fmax; out->Frms = nsim > 0 ? sqrt(h.FF / nsim) : 0.0;
    out->P = 0.0; out->dt = dp->eta; out->alpha = dp->mu;
    out->launches = launches; out->sweep_launches = sweeps; out->gpu_ms = ms;
    if (dp->report_energy) {
        rc = lq_energy(c, &out->energy);
        if (rc != LQ_OK) return rc;
    }
    return LQ_OK;
}

}  // extern "C"

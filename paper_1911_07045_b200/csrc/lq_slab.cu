// lq_slab.cu -- domain decomposition into z-slabs (section III.B: "the simulation
// domain is divided into rectilinear sub-domains ... after each step the sites on the faces of neighbouring
// sub-domains are communicated ... and the scalar quantities of the minimiser are reduced over all ranks").
//
// A sub-domain is an ordinary context whose lattice is the slab [z0, z0 + nz) of a global Lx x Ly x Lz lattice and
// whose geometry has zopen = 1: nothing wraps in z, no kernel writes z ghost images, and the two z ghost planes on
// each side hold the neighbour slabs' boundary planes.  One FIRE step of the decomposed lattice is
//     every sub-domain: the same fused sweep as the single-domain path, with the schedule update deferred
//     halo exchange:    2 planes of (q, vc [, F]) per face (nearest and next-nearest sites: the recompute sweep
//                       reads q two sites deep)
//     reduction:        the per-CTA partials of all sub-domains, in a fixed order -> (P, |F|^2, |v|^2, max|F|)
//                       -> the same schedule update in every sub-domain's device scalars
// Two drivers share these pieces.  lq_slabs_* runs N sub-domains of one process on one GPU (device-to-device plane
// copies, one reduction kernel over all sub-domains' partials): this is what the B200 tests run against the
// oracle.  lq_halo_export / lq_halo_import / lq_fire_step_local / lq_fire_step_commit are the transport-agnostic
// pieces for one rank per GPU (the Python driver moves the packages and the 6-double rows with
// torch.distributed / NCCL); that route is unmeasured on hardware here (one GPU per lease).
#include "lq_ctx.cuh"

#include <cmath>
#include <cstring>
#include <new>
#include <vector>

namespace {

#define LQ_CUDA(c, call)                                                                             \
    do {                                                                                             \
        cudaError_t e_ = (call);                                                                     \
        if (e_ != cudaSuccess)                                                                       \
            return fail((c), e_ == cudaErrorMemoryAllocation ? LQ_ERR_NOMEM : LQ_ERR_CUDA,           \
                        std::string(#call) + ": " + cudaGetErrorString(e_));                         \
    } while (0)

bool stored_path(const lq_ctx *c) { return lq_three(c->ph) || c->fire_path == 2; }

// the 5-component fields a halo package of kind `what` carries, in order
int halo_fields(lq_ctx *c, int what, double *out[3]) {
    if (what == LQ_HALO_Q) { out[0] = c->q[c->cur]; return 1; }
    const int b = c->fire_open ? c->fire_buf : c->cur;
    int n = 0;
    out[n++] = c->q[b];
    out[n++] = c->v[b];
    if (stored_path(c)) out[n++] = c->F[b];
    return n;
}

// padded plane index of the first of the two planes a face exports / imports
int export_plane(const lq_ctx *c, int face) { return face == 0 ? LQ_GH : c->g.Lz; }            // z = 0,1 | nz-2,nz-1
int import_plane(const lq_ctx *c, int face) { return face == 0 ? 0 : c->g.Lz + LQ_GH; }        // z = -2,-1 | nz,nz+1

bool same_group(lq_ctx **s, int n, std::string *why) {
    for (int i = 0; i < n; ++i) {
        if (!s[i] || !s[i]->g.zopen) { *why = "every member must be a context made by lq_create_slab"; return false; }
        if (s[i]->g.Lx != s[0]->g.Lx || s[i]->g.Ly != s[0]->g.Ly || s[i]->Lz_global != s[0]->Lz_global ||
            s[i]->device != s[0]->device) { *why = "members differ in Lx, Ly, global Lz or device"; return false; }
    }
    int z = s[0]->z0, tot = 0;
    for (int i = 0; i < n; ++i) {
        if (s[i]->z0 != z) { *why = "slabs must be listed in z order and tile the lattice"; return false; }
        z += s[i]->g.Lz; tot += s[i]->g.Lz;
    }
    if (tot != s[0]->Lz_global || s[0]->z0 != 0) { *why = "slabs must tile [0, Lz) starting at z0 = 0"; return false; }
    return true;
}

int fire_begin(lq_ctx *c, long max_steps, double force_tol, const lq_fire_params *fp) {
    if (!c->g.zopen) return fail(c, LQ_ERR_STATE, "lq_fire_begin: not a sub-domain context (use lq_fire_minimize)");
    if (!fp) return fail(c, LQ_ERR_ARG, "lq_fire_begin: NULL params");
    if (!c->has_Q) return fail(c, LQ_ERR_STATE, "lq_fire_begin: no Q has been set");
    if (c->fire_path == 1) return fail(c, LQ_ERR_STATE, "lq_fire_begin: sub-domains run the fused sweeps only (fire_path 0 or 2)");
    if (!(fp->dt0 > 0.0) || !(fp->dtmax >= fp->dt0) || !(fp->alpha0 >= 0.0 && fp->alpha0 <= 1.0) ||
        !(fp->finc >= 1.0) || !(fp->fdec > 0.0 && fp->fdec <= 1.0) || !(fp->falpha > 0.0 && fp->falpha <= 1.0) ||
        fp->Nmin < 0 || (fp->integrator != 0 && fp->integrator != 1) || max_steps < 0 || !(force_tol >= 0.0))
        return fail(c, LQ_ERR_ARG, "lq_fire_begin: bad FIRE parameter");
    const bool euler = fp->integrator == 1, stored = stored_path(c);
    int rc;
    for (int b = 0; b < 2; ++b) {
        if ((rc = lq_ensure_field(c, &c->q[b])) != LQ_OK) return rc;
        if ((rc = lq_ensure_field(c, &c->v[b])) != LQ_OK) return rc;
        if (stored && (rc = lq_ensure_field(c, &c->F[b])) != LQ_OK) return rc;
    }
    c->fire_fc = LqFireConsts{fp->dt0, fp->dtmax, fp->alpha0, fp->finc, fp->fdec, fp->falpha, force_tol, fp->Nmin,
                              (long long)max_steps, euler ? 1 : 0};
    LqFireScalars h;
    memset(&h, 0, sizeof(h));
    h.dt = fp->dt0; h.alpha = fp->alpha0; h.init = (stored && !euler) ? 1 : 0;
    LQ_CUDA(c, cudaMemcpyAsync(&c->dsc[0], &h, sizeof(h), cudaMemcpyHostToDevice, c->stream));
    c->fire_launches = 0; c->fire_sweeps = 0;
    rc = lq_sweep_prepare(&c->sweep, stored, c->g, c->ph, fields_of(c), c->q, c->v, c->F, c->stream, &c->fire_launches, c->err,
                          c->rc_chunks);
    if (rc != LQ_OK) return rc;
    if (!c->dtot) LQ_CUDA(c, cudaMalloc(&c->dtot, 6 * sizeof(double)));
    if (!c->dsegs) LQ_CUDA(c, cudaMalloc(&c->dsegs, 8 * sizeof(LqPartialSeg)));
    if (!c->dscptr) {
        LQ_CUDA(c, cudaMalloc(&c->dscptr, sizeof(LqFireScalars *)));
        LqFireScalars *p = &c->dsc[0];
        LQ_CUDA(c, cudaMemcpyAsync(c->dscptr, &p, sizeof(p), cudaMemcpyHostToDevice, c->stream));
    }
    c->fire_cur0 = c->cur; c->fire_buf = c->cur; c->fire_open = true; c->fire_last_first = false;
    LQ_CUDA(c, cudaEventRecord(c->ev0, c->stream));
    return LQ_OK;
}

// sweeps a whole run enqueues at most (see lq_sweep_run): recompute + velocity Verlet: max(max_steps, 1); else +1
long fire_total_sweeps(const lq_ctx *c) {
    const bool extra = stored_path(c) || c->fire_fc.euler;
    return extra ? (long)c->fire_fc.max_steps + 1 : ((long)c->fire_fc.max_steps > 0 ? (long)c->fire_fc.max_steps : 1);
}

bool has_fixup(const lq_ctx *c) { return stored_path(c) && c->flags_active; }

// one deferred sweep (without its fix-up launch, which needs the neighbours' new q' across the faces first)
int fire_sweep(lq_ctx *c) {
    const bool stored = stored_path(c);
    const bool first = !stored && !c->fire_fc.euler && c->fire_sweeps == 0;
    const int in = (int)((c->fire_cur0 + c->fire_sweeps) & 1);
    int rc = lq_sweep_step(c->sweep, stored, c->g, c->ph, fields_of(c), c->q, c->v, c->F, in, c->dsc, c->fire_fc, first, true,
                           c->stream, c->err, 1);
    if (rc != LQ_OK) return rc;
    c->fire_sweeps += 1;
    c->fire_launches += 1;
    c->fire_buf = in ^ 1;
    c->fire_last_first = first;
    c->fire_sweep_pending = true;
    return LQ_OK;
}

// the rest of the step on this sub-domain: the fix-up launch where the path has one; the partial-sum segments the
// step left behind go to seg[] (their number through *nseg)
int fire_finish(lq_ctx *c, LqPartialSeg seg[3], int *nseg) {
    if (!c->fire_sweep_pending) return fail(c, LQ_ERR_STATE, "lq_fire_step_finish: no sweep is pending (call lq_fire_step_local)");
    const bool stored = stored_path(c);
    const LqFields f = fields_of(c);
    if (has_fixup(c)) {
        const int in = c->fire_buf ^ 1;
        int rc = lq_sweep_step(c->sweep, stored, c->g, c->ph, f, c->q, c->v, c->F, in, c->dsc, c->fire_fc, false, true, c->stream,
                               c->err, 2);
        if (rc != LQ_OK) return rc;
        c->fire_launches += 1;
    }
    *nseg = lq_sweep_segments(c->sweep, stored, f.flags != nullptr, c->fire_last_first, seg);
    c->fire_sweep_pending = false;
    return LQ_OK;
}

// the segment table of a step on the device: it changes only between the first sweep and the rest of a run, so it is
// uploaded when it differs from what the device copy already holds, not every step
cudaError_t upload_segments(lq_ctx *c, const LqPartialSeg *seg, int nseg) {
    if (nseg == c->hnseg && memcmp(seg, c->hsegs, nseg * sizeof(LqPartialSeg)) == 0) return cudaSuccess;
    // pageable source: staged before the call returns, so hsegs may change right after
    const cudaError_t e = cudaMemcpyAsync(c->dsegs, seg, nseg * sizeof(LqPartialSeg), cudaMemcpyHostToDevice, c->stream);
    if (e != cudaSuccess) { c->hnseg = -1; return e; }
    memset(c->hsegs, 0, sizeof(c->hsegs));
    memcpy(c->hsegs, seg, nseg * sizeof(LqPartialSeg));
    c->hnseg = nseg;
    return cudaSuccess;
}

// a step-wise run given up half way: leave the context as it was before lq_fire_begin (live buffer, no open run)
void fire_abort(lq_ctx *c) {
    if (!c->fire_open) return;
    c->fire_open = false;
    c->fire_sweep_pending = false;
    c->cur = c->fire_cur0;
}

int fire_end(lq_ctx *c, lq_fire_report *out) {
    if (!c->fire_open) return fail(c, LQ_ERR_STATE, "lq_fire_end: no step-wise FIRE run is open");
    LqFireScalars h;
    LQ_CUDA(c, cudaEventRecord(c->ev1, c->stream));
    LQ_CUDA(c, cudaMemcpyAsync(&h, &c->dsc[0], sizeof(h), cudaMemcpyDeviceToHost, c->stream));
    LQ_CUDA(c, cudaStreamSynchronize(c->stream));
    LQ_CUDA(c, cudaGetLastError());
    const bool extra = stored_path(c) || c->fire_fc.euler;
    long flips = (long)h.step + (extra ? 1 : 0);
    if (flips > c->fire_sweeps) flips = c->fire_sweeps;          // run closed early by the caller
    c->cur = (int)((c->fire_cur0 + flips) & 1);
    c->fire_open = false;
    c->v_valid = h.step > 0;
    const bool pending = !h.converged && h.step > 0 && !(c->fire_fc.euler && h.step >= c->fire_fc.max_steps);
    c->v_mix_a = pending ? h.mix_a : 1.0;
    c->v_mix_b = pending ? h.mix_b : 0.0;
    if (out) {
        memset(out, 0, sizeof(*out));
        float ms = 0.f;
        cudaEventElapsedTime(&ms, c->ev0, c->ev1);
        // Frms is a property of the whole lattice: the caller divides by the global number of simulated sites
        const double nsim = (double)(c->flags_active ? c->n_class[0] + c->n_class[1] : (unsigned long long)c->g.N);
        out->steps = (long)h.step; out->converged = h.converged;
        out->Fmax = h.Fmax; out->Frms = nsim > 0 ? sqrt(h.FF / nsim) : 0.0;
        out->P = h.P; out->dt = h.dt; out->alpha = h.alpha;
        out->launches = c->fire_launches; out->sweep_launches = c->fire_sweeps; out->gpu_ms = ms;
    }
    return LQ_OK;
}

cudaError_t copy_planes(lq_ctx *dst, int dplane, double *dfield, lq_ctx *src, int splane, const double *sfield,
                        cudaStream_t st) {
    const size_t sz = (size_t)dst->g.sz;
    return cudaMemcpy2DAsync(dfield + sz * dplane, (size_t)dst->g.NP * sizeof(double), sfield + sz * splane,
                             (size_t)src->g.NP * sizeof(double), 2 * sz * sizeof(double), 5, cudaMemcpyDeviceToDevice, st);
}

int slabs_exchange(lq_ctx **s, int n, int what, cudaStream_t st) {
    for (int i = 0; i < n; ++i) {
        lq_ctx *lo = s[(i + n - 1) % n], *hi = s[(i + 1) % n], *c = s[i];
        double *fc[3], *fl[3], *fh[3];
        const int nf = halo_fields(c, what, fc);
        halo_fields(lo, what, fl);
        halo_fields(hi, what, fh);
        for (int k = 0; k < nf; ++k) {
            if (!fc[k] || !fl[k] || !fh[k]) return fail(c, LQ_ERR_STATE, "lq_slabs_exchange: field not allocated (set Q first)");
            // my low ghost planes <- the upper two planes of the slab below; my high ghost planes <- the lower two above
            LQ_CUDA(c, copy_planes(c, import_plane(c, 0), fc[k], lo, export_plane(lo, 1), fl[k], st));
            LQ_CUDA(c, copy_planes(c, import_plane(c, 1), fc[k], hi, export_plane(hi, 0), fh[k], st));
        }
    }
    return LQ_OK;
}

}  // namespace

extern "C" {

int lq_create_slab(int Lx, int Ly, int Lz_global, int z0, int nz, double A, double B, double C, double L1, double L2,
                   double L3, lq_ctx **out) {
    if (!out) return fail(nullptr, LQ_ERR_ARG, "lq_create_slab: out is NULL");
    *out = nullptr;
    if (Lz_global < 4 || z0 < 0 || nz < 4 || z0 + nz > Lz_global)
        return fail(nullptr, LQ_ERR_ARG, "lq_create_slab: need Lz >= 4, nz >= 4 and [z0, z0 + nz) inside [0, Lz)");
    int rc = lq_create(Lx, Ly, nz, A, B, C, L1, L2, L3, out);
    if (rc != LQ_OK) return rc;
    (*out)->g.zopen = 1;
    (*out)->Lz_global = Lz_global;
    (*out)->z0 = z0;
    return LQ_OK;
}

int lq_set_sites_ext(lq_ctx *c, const uint8_t *mask_ext, const uint8_t *kind_ext, const double *W_ext, const double *axis_ext,
                     int where) {
    if (!c) return LQ_ERR_ARG;
    DeviceGuard dg(c);
    if (!c->g.zopen) return fail(c, LQ_ERR_STATE, "lq_set_sites_ext: not a sub-domain context");
    if (bad_where(where) || !mask_ext) return fail(c, LQ_ERR_ARG, "lq_set_sites_ext: bad argument");
    if (kind_ext && (!W_ext || !axis_ext)) return fail(c, LQ_ERR_ARG, "lq_set_sites_ext: kind given without W / axis");
    const LqGeom &g = c->g;
    cudaStream_t st = c->stream;
    const size_t next = (size_t)g.Lx * g.Ly * (g.Lz + 6);
    lq_sweep_invalidate(c->sweep);
    lq_descent_invalidate(c->descent);
    // the dense mask with its 3-plane margin on the device
    uint8_t *dmask = nullptr, *dkind = nullptr;
    struct FreeOnExit { uint8_t *&p; ~FreeOnExit() { cudaFree(p); p = nullptr; } } free_dmask{dmask};   // every return path
    LQ_CUDA(c, cudaMalloc(&dmask, next));
    cudaError_t e = cudaMemcpyAsync(dmask, mask_ext, next, cudaMemcpyDefault, st);
    int bad[2] = {0, 0};
    if (e == cudaSuccess) e = cudaMemsetAsync(c->dbad, 0, 2 * sizeof(int), st);
    if (e == cudaSuccess) lq_launch_check_dense_u8_max(dmask, (long long)next, 1, c->dbad, st);
    if (e == cudaSuccess && kind_ext) {
        e = cudaMalloc(&dkind, next);
        if (e == cudaSuccess) e = cudaMemcpyAsync(dkind, kind_ext, next, cudaMemcpyDefault, st);
        if (e == cudaSuccess) lq_launch_check_dense_u8_max(dkind, (long long)next, 2, c->dbad + 1, st);
    }
    if (e == cudaSuccess) e = cudaMemcpyAsync(bad, c->dbad, 2 * sizeof(int), cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e != cudaSuccess || bad[0] || bad[1]) {
        cudaFree(dkind);
        c->flags_active = false; c->anch_active = false;
        c->n_class[0] = (unsigned long long)g.N; c->n_class[1] = c->n_class[2] = 0;
        if (e != cudaSuccess) return fail(c, LQ_ERR_CUDA, std::string("lq_set_sites_ext: ") + cudaGetErrorString(e));
        return fail(c, LQ_ERR_ARG, bad[0] ? "lq_set_sites_ext: mask value > 1 (sites reset to all bulk)"
                                          : "lq_set_sites_ext: anch_kind value > 2 (sites reset to all bulk)");
    }
    cudaFree(dkind);
    if (!c->flags) LQ_CUDA(c, cudaMalloc(&c->flags, (size_t)g.NP));
    LQ_CUDA(c, cudaMemsetAsync(c->flags, 0xFC, (size_t)g.NP, st));
    lq_launch_classify_ext(g, dmask, c->flags, st);
    lq_launch_fill_ghosts_u8(g, c->flags, st);                 // x / y ghosts of every plane, z ghost planes included
    LQ_CUDA(c, cudaMemsetAsync(c->dcounts, 0, 3 * sizeof(unsigned long long), st));
    lq_launch_count_classes(g, c->flags, c->dcounts, st);
    if (kind_ext) {
        if (!c->kind) LQ_CUDA(c, cudaMalloc(&c->kind, (size_t)g.NP));
        if (!c->W) LQ_CUDA(c, cudaMalloc(&c->W, (size_t)g.NP * sizeof(double)));
        if (!c->axis) LQ_CUDA(c, cudaMalloc(&c->axis, (size_t)3 * g.NP * sizeof(double)));
        LQ_CUDA(c, cudaMemsetAsync(c->kind, 0, (size_t)g.NP, st));
        LQ_CUDA(c, cudaMemsetAsync(c->W, 0, (size_t)g.NP * sizeof(double), st));
        LQ_CUDA(c, cudaMemsetAsync(c->axis, 0, (size_t)3 * g.NP * sizeof(double), st));
        // ext planes 1 .. nz+4 (z = -2 .. nz+1) -> every padded plane
        LQ_CUDA(c, lq_copy_box(g, c->kind, kind_ext, 1, 1, true, st, 0, g.Pz, 1, g.Lz + 6));
        LQ_CUDA(c, lq_copy_box(g, c->W, W_ext, sizeof(double), 1, true, st, 0, g.Pz, 1, g.Lz + 6));
        LQ_CUDA(c, lq_copy_box(g, c->axis, axis_ext, sizeof(double), 3, true, st, 0, g.Pz, 1, g.Lz + 6));
        lq_launch_fill_ghosts_u8(g, c->kind, st);
        lq_launch_fill_ghosts_f64(g, c->W, 1, st);
        lq_launch_fill_ghosts_f64(g, c->axis, 3, st);
    }
    // a slab with no object of its own may still touch one across a face: any flag byte other than "bulk, all six
    // neighbours simulated" on the padded array (ghost planes included) switches the masked kernels on
    int any = 0;
    LQ_CUDA(c, cudaMemsetAsync(c->dbad, 0, sizeof(int), st));
    lq_launch_check_dense_u8_ne(c->flags, (long long)g.NP, 0xFC, c->dbad, st);
    LQ_CUDA(c, cudaMemcpyAsync(&any, c->dbad, sizeof(int), cudaMemcpyDeviceToHost, st));
    LQ_CUDA(c, cudaMemcpyAsync(c->n_class, c->dcounts, 3 * sizeof(unsigned long long), cudaMemcpyDeviceToHost, st));
    LQ_CUDA(c, cudaStreamSynchronize(st));
    LQ_CUDA(c, cudaGetLastError());
    c->flags_active = any != 0;
    c->anch_active = kind_ext != nullptr && any != 0;
    return LQ_OK;
}

int lq_halo_bytes(lq_ctx *c, int what, size_t *bytes) {
    if (!c || !bytes) return LQ_ERR_ARG;
    if (what != LQ_HALO_Q && what != LQ_HALO_STATE) return fail(c, LQ_ERR_ARG, "lq_halo_bytes: bad `what`");
    const int nf = what == LQ_HALO_Q ? 1 : (stored_path(c) ? 3 : 2);
    *bytes = (size_t)nf * 5 * 2 * (size_t)c->g.sz * sizeof(double);
    return LQ_OK;
}

static int halo_move(lq_ctx *c, int what, int face, void *buf, int where, bool do_export) {
    if (!c) return LQ_ERR_ARG;
    DeviceGuard dg(c);
    if (!c->g.zopen) return fail(c, LQ_ERR_STATE, "lq_halo_*: not a sub-domain context");
    if (!buf || bad_where(where) || (face != 0 && face != 1) || (what != LQ_HALO_Q && what != LQ_HALO_STATE))
        return fail(c, LQ_ERR_ARG, "lq_halo_*: bad argument");
    if (!c->has_Q) return fail(c, LQ_ERR_STATE, "lq_halo_*: no Q has been set");
    double *f[3];
    const int nf = halo_fields(c, what, f);
    const size_t sz = (size_t)c->g.sz, row = 2 * sz * sizeof(double);
    const int plane = do_export ? export_plane(c, face) : import_plane(c, face);
    for (int k = 0; k < nf; ++k) {
        if (!f[k]) return fail(c, LQ_ERR_STATE, "lq_halo_*: field not allocated");
        char *pk = (char *)buf + (size_t)k * 5 * row;
        double *fld = f[k] + sz * plane;
        if (do_export) LQ_CUDA(c, cudaMemcpy2DAsync(pk, row, fld, (size_t)c->g.NP * sizeof(double), row, 5, cudaMemcpyDefault, c->stream));
        else LQ_CUDA(c, cudaMemcpy2DAsync(fld, (size_t)c->g.NP * sizeof(double), pk, row, row, 5, cudaMemcpyDefault, c->stream));
    }
    if (where == LQ_HOST) LQ_CUDA(c, cudaStreamSynchronize(c->stream));
    return LQ_OK;
}
int lq_halo_export(lq_ctx *c, int what, int face, void *buf, int where) { return halo_move(c, what, face, buf, where, true); }
int lq_halo_import(lq_ctx *c, int what, int face, const void *buf, int where) {
    return halo_move(c, what, face, const_cast<void *>(buf), where, false);
}

int lq_fire_begin(lq_ctx *c, long max_steps, double force_tol, const lq_fire_params *fp) {
    if (!c) return LQ_ERR_ARG;
    DeviceGuard dg(c);
    return fire_begin(c, max_steps, force_tol, fp);
}

int lq_fire_step_local(lq_ctx *c) {
    if (!c) return LQ_ERR_ARG;
    DeviceGuard dg(c);
    if (!c->fire_open) return fail(c, LQ_ERR_STATE, "lq_fire_step_local: call lq_fire_begin first");
    if (c->fire_sweep_pending) return fail(c, LQ_ERR_STATE, "lq_fire_step_local: the previous sweep was not finished (lq_fire_step_finish)");
    return fire_sweep(c);
}

int lq_fire_step_finish(lq_ctx *c, double *tot6, int where, int *exchange_again) {
    if (!c) return LQ_ERR_ARG;
    DeviceGuard dg(c);
    if (!c->fire_open) return fail(c, LQ_ERR_STATE, "lq_fire_step_finish: call lq_fire_begin first");
    if (!tot6 || bad_where(where)) return fail(c, LQ_ERR_ARG, "lq_fire_step_finish: bad argument");
    LqPartialSeg seg[3];
    int nseg = 0;
    int rc = fire_finish(c, seg, &nseg);
    if (rc != LQ_OK) return rc;
    LQ_CUDA(c, upload_segments(c, seg, nseg));
    lq_launch_reduce_partials(c->dsegs, nseg, c->dtot, c->stream);
    LQ_CUDA(c, cudaMemcpyAsync(tot6, c->dtot, 6 * sizeof(double), cudaMemcpyDefault, c->stream));
    if (where == LQ_HOST) LQ_CUDA(c, cudaStreamSynchronize(c->stream));
    if (exchange_again) *exchange_again = has_fixup(c) ? 1 : 0;
    return LQ_OK;
}

int lq_fire_step_commit(lq_ctx *c, const double *tot, int nrank, int where) {
    if (!c) return LQ_ERR_ARG;
    DeviceGuard dg(c);
    if (!c->fire_open) return fail(c, LQ_ERR_STATE, "lq_fire_step_commit: call lq_fire_begin first");
    if (!tot || nrank < 1 || bad_where(where)) return fail(c, LQ_ERR_ARG, "lq_fire_step_commit: bad argument");
    const double *dt = tot;
    if (where == LQ_HOST) {
        if ((size_t)nrank * 6 * sizeof(double) > c->scratch_len) {
            cudaFree(c->scratch); c->scratch = nullptr; c->scratch_len = 0;
            LQ_CUDA(c, cudaMalloc(&c->scratch, (size_t)nrank * 6 * sizeof(double)));
            c->scratch_len = (size_t)nrank * 6 * sizeof(double);
        }
        LQ_CUDA(c, cudaMemcpyAsync(c->scratch, tot, (size_t)nrank * 6 * sizeof(double), cudaMemcpyHostToDevice, c->stream));
        LQ_CUDA(c, cudaStreamSynchronize(c->stream));    // pinned host rows are read asynchronously: free to reuse on return
        dt = (const double *)c->scratch;
    }
    lq_launch_advance(dt, nrank, c->dscptr, 1, c->fire_fc, c->fire_last_first ? 1 : 0, c->stream);
    LQ_CUDA(c, cudaGetLastError());
    return LQ_OK;
}

int lq_fire_peek(lq_ctx *c, lq_fire_report *out) {
    if (!c) return LQ_ERR_ARG;
    DeviceGuard dg(c);
    if (!c->fire_open || !out) return fail(c, LQ_ERR_STATE, "lq_fire_peek: no step-wise FIRE run is open");
    LqFireScalars h;
    LQ_CUDA(c, cudaMemcpyAsync(&h, &c->dsc[0], sizeof(h), cudaMemcpyDeviceToHost, c->stream));
    LQ_CUDA(c, cudaStreamSynchronize(c->stream));
    memset(out, 0, sizeof(*out));
    out->steps = (long)h.step; out->converged = h.converged; out->Fmax = h.Fmax; out->P = h.P; out->dt = h.dt; out->alpha = h.alpha;
    out->launches = c->fire_launches; out->sweep_launches = c->fire_sweeps;
    return LQ_OK;
}

int lq_fire_end(lq_ctx *c, lq_fire_report *out) {
    if (!c) return LQ_ERR_ARG;
    DeviceGuard dg(c);
    return fire_end(c, out);
}

int lq_slabs_exchange(lq_ctx **slabs, int n, int what) {
    if (!slabs || n < 1 || !slabs[0]) return LQ_ERR_ARG;
    DeviceGuard dg(slabs[0]);
    std::string why;
    if (!same_group(slabs, n, &why)) return fail(slabs[0], LQ_ERR_ARG, "lq_slabs_exchange: " + why);
    if (what != LQ_HALO_Q && what != LQ_HALO_STATE) return fail(slabs[0], LQ_ERR_ARG, "lq_slabs_exchange: bad `what`");
    cudaStream_t st = slabs[0]->stream;
    for (int i = 0; i < n; ++i)
        if (!slabs[i]->has_Q) return fail(slabs[0], LQ_ERR_STATE, "lq_slabs_exchange: every slab needs lq_set_Q first");
    int rc = slabs_exchange(slabs, n, what, st);
    if (rc != LQ_OK) return rc;
    LQ_CUDA(slabs[0], cudaStreamSynchronize(st));
    return LQ_OK;
}

int lq_slabs_fire_minimize(lq_ctx **slabs, int n, long max_steps, double force_tol, const lq_fire_params *fp,
                           lq_fire_report *out) {
    if (!slabs || n < 1 || !slabs[0]) return LQ_ERR_ARG;
    lq_ctx *c0 = slabs[0];
    DeviceGuard dg(c0);
    std::string why;
    if (!same_group(slabs, n, &why)) return fail(c0, LQ_ERR_ARG, "lq_slabs_fire_minimize: " + why);
    if (!fp || !out) return fail(c0, LQ_ERR_ARG, "lq_slabs_fire_minimize: NULL params / report");
    cudaStream_t st = c0->stream;
    for (int i = 0; i < n; ++i) {
        if (slabs[i]->stream != st) return fail(c0, LQ_ERR_ARG, "lq_slabs_fire_minimize: all slabs must use one stream");
        if (stored_path(slabs[i]) != stored_path(c0)) return fail(c0, LQ_ERR_ARG, "lq_slabs_fire_minimize: mixed sweep paths");
    }
    int rc;
    if ((rc = slabs_exchange(slabs, n, LQ_HALO_Q, st)) != LQ_OK) return rc;       // ghosts of the initial state
    LqFireScalars **dscs = nullptr;
    double *drows = nullptr;
    // every exit below goes through one of these two: device tables freed; on failure every slab's run closed too
    auto cleanup = [&]() { cudaFree(dscs); cudaFree(drows); dscs = nullptr; drows = nullptr; };
    auto give_up = [&](int code, lq_ctx *who) {
        if (who && who != c0) c0->err = who->err;
        for (int i = 0; i < n; ++i) fire_abort(slabs[i]);
        cleanup();
        return code;
    };
    for (int i = 0; i < n; ++i)
        if ((rc = fire_begin(slabs[i], max_steps, force_tol, fp)) != LQ_OK) return give_up(rc, slabs[i]);
    // device tables: every slab's scalars; one row of reductions per slab (combined in slab order by the advance
    // kernel: the same arithmetic as the one-rank-per-GPU protocol, so both give bit-identical trajectories)
    std::vector<LqFireScalars *> scs(n);
    for (int i = 0; i < n; ++i) scs[i] = &slabs[i]->dsc[0];
    if (cudaMalloc(&dscs, n * sizeof(LqFireScalars *)) != cudaSuccess || cudaMalloc(&drows, (size_t)6 * n * sizeof(double)) != cudaSuccess)
        return give_up(fail(c0, LQ_ERR_NOMEM, "lq_slabs_fire_minimize: cudaMalloc failed"), nullptr);
    if (cudaMemcpyAsync(dscs, scs.data(), n * sizeof(LqFireScalars *), cudaMemcpyHostToDevice, st) != cudaSuccess)
        return give_up(fail(c0, LQ_ERR_CUDA, "lq_slabs_fire_minimize: upload of the scalar table failed"), nullptr);
    bool any_fixup = false;
    for (int i = 0; i < n; ++i) any_fixup |= has_fixup(slabs[i]);
    const long total = fire_total_sweeps(c0);
    long done = 0;
    LqFireScalars h;
    memset(&h, 0, sizeof(h));
    while (done < total) {
        const long chunk = force_tol > 0.0 ? 100 : total;
        const long m = (total - done) < chunk ? (total - done) : chunk;
        for (long s = 0; s < m; ++s) {
            for (int i = 0; i < n; ++i)
                if ((rc = fire_sweep(slabs[i])) != LQ_OK) return give_up(rc, slabs[i]);
            // the new state's boundary planes to the neighbours; where a fix-up launch follows (it evaluates the force
            // of the sites next to objects on q', across the slab faces too) it changes v and F there: exchange again
            if ((rc = slabs_exchange(slabs, n, LQ_HALO_STATE, st)) != LQ_OK) return give_up(rc, nullptr);
            for (int i = 0; i < n; ++i) {
                lq_ctx *c = slabs[i];
                LqPartialSeg sg[3];
                int ns = 0;
                if ((rc = fire_finish(c, sg, &ns)) != LQ_OK) return give_up(rc, c);
                if (upload_segments(c, sg, ns) != cudaSuccess)
                    return give_up(fail(c0, LQ_ERR_CUDA, "lq_slabs_fire_minimize: upload of the segment table failed"), nullptr);
                lq_launch_reduce_partials(c->dsegs, ns, drows + 6 * i, st);
            }
            lq_launch_advance(drows, n, dscs, n, c0->fire_fc, c0->fire_last_first ? 1 : 0, st);
            if (any_fixup && (rc = slabs_exchange(slabs, n, LQ_HALO_STATE, st)) != LQ_OK) return give_up(rc, nullptr);
        }
        done += m;
        if (force_tol > 0.0) {
            if (cudaMemcpyAsync(&h, &c0->dsc[0], sizeof(h), cudaMemcpyDeviceToHost, st) != cudaSuccess || cudaStreamSynchronize(st) != cudaSuccess)
                return give_up(fail(c0, LQ_ERR_CUDA, "lq_slabs_fire_minimize: stream error"), nullptr);
            if (h.converged) break;
        }
    }
    double nsim = 0.0;
    lq_fire_report rep;
    for (int i = 0; i < n; ++i) {
        if ((rc = fire_end(slabs[i], i == 0 ? out : &rep)) != LQ_OK) return give_up(rc, slabs[i]);
        nsim += (double)(slabs[i]->flags_active ? slabs[i]->n_class[0] + slabs[i]->n_class[1] : (unsigned long long)slabs[i]->g.N);
        if (i > 0) { out->launches += rep.launches; out->sweep_launches += rep.sweep_launches; }
    }
    cleanup();
    // the final state's ghost planes (a step the stop test discarded leaves the live buffer's ghosts untouched)
    if ((rc = slabs_exchange(slabs, n, LQ_HALO_Q, st)) != LQ_OK) return rc;
    LQ_CUDA(c0, cudaStreamSynchronize(st));
    // Frms over the whole lattice: fire_end divided |F|^2 (a global sum already) by the slab's own site count
    const double nsim0 = (double)(c0->flags_active ? c0->n_class[0] + c0->n_class[1] : (unsigned long long)c0->g.N);
    out->Frms = nsim > 0 ? out->Frms * sqrt(nsim0 / nsim) : 0.0;
    out->launches += out->sweep_launches + out->sweep_launches / n;   // per step: one reduction kernel per slab + one advance kernel
    if (fp->report_energy) {
        double e = 0.0;
        for (int i = 0; i < n; ++i) {
            double ei = 0.0;
            if ((rc = lq_energy(slabs[i], &ei)) != LQ_OK) return rc;
            e += ei;
        }
        out->energy = e;
    }
    return LQ_OK;
}

}  // extern "C"

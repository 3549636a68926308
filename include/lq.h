/*
 * lq.h -- C ABI of liblq.so: the B200 (sm_100a) hot path of lattice Landau-de Gennes
 * Q-tensor minimisation with FIRE (arXiv:1911.07045, Sussman & Beller, "openQmin").
 *
 * Citations: "PAPER.md:<line>" = /root/reference/PAPER.md with the section / equation
 * the line falls in; "DESIGN.md Rn" = reading n of a silent or garbled passage.
 *
 * Conventions (all calls)
 *   - Lattice: Lx x Ly x Lz cubic lattice, spacing 1, site index s = x + Lx*(y + Ly*z),
 *     N = Lx*Ly*Lz.  Index arithmetic is periodic in x, y and z; walls are layers of
 *     object sites supplied through lq_set_sites (R14).
 *   - Fields: fp64, structure of arrays [5][N], component order (xx, xy, xz, yy, yz)
 *     (PAPER.md:173); Qzz = -Qxx - Qyy is implied.  Everything is in the paper's lattice
 *     units (energy density / |A|-scale, lengths / lattice spacing).
 *   - `where` says where the CALLER's buffer lives: LQ_HOST (pageable or pinned host
 *     memory) or LQ_DEVICE (a device pointer on the context's GPU, e.g. a torch tensor's
 *     data_ptr()).  set_* copy in, get_* / lq_forces copy out; the library never keeps a
 *     caller pointer after the call returns.  Copies and kernels are enqueued on the
 *     context's stream (lq_set_stream; default: the legacy default stream) and every call
 *     that returns data to the host synchronises that stream before returning.
 *   - Ownership: the library owns the context and every internal device buffer; the
 *     caller owns every pointer it passes.
 *   - Errors: every int-returning call returns LQ_OK or a negative LQ_ERR_*; nothing
 *     throws or aborts across the ABI.  lq_last_error gives a message for the last
 *     failing call on that context.  There is NO CPU fallback: without a usable CUDA
 *     device lq_create fails with LQ_ERR_CUDA.
 */
#ifndef LQ_H
#define LQ_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct lq_ctx lq_ctx; /* opaque; owned by the library */

enum { LQ_OK = 0, LQ_ERR_ARG = -1, LQ_ERR_STATE = -2, LQ_ERR_CUDA = -3, LQ_ERR_NOMEM = -4 };
enum { LQ_HOST = 0, LQ_DEVICE = 1 };
enum { LQ_SITE_LC = 0, LQ_SITE_OBJECT = 1 }; /* values of the input mask */
enum { LQ_ANCH_NONE = 0, LQ_ANCH_ORIENTED = 1 /* Eq. 14 */, LQ_ANCH_DEGENERATE_PLANAR = 2 /* Eq. 15 */ };

/* packed site byte returned by lq_get_flags ("integer type"; R8):
 *   bits 0-1: class  0 bulk, 1 boundary (simulated, >= 1 of its 6 face neighbours is an
 *             object), 2 object (not simulated)
 *   bit 2: site +x is simulated   bit 3: -x   bit 4: +y   bit 5: -y   bit 6: +z   bit 7: -z
 *   (neighbour bits are set the same way at object sites). */
enum { LQ_CLASS_BULK = 0, LQ_CLASS_BOUNDARY = 1, LQ_CLASS_OBJECT = 2 };

/* Create a context for an Lx x Ly x Lz lattice with the bulk constants A, B, C of Eq. 5
 * and the distortion constants L1, L2, L3 of Eq. 10 (L4 = L6 = 0;
 * L2 = L3 = 0 selects the one-constant form Eq. 11).  All sites start as bulk
 * liquid crystal with no anchoring and Q undefined.  The context computes
 * S0 = (-B + sqrt(B^2 - 24 A C)) / (6 C) (Eq. 7) for the anchoring terms.
 * Errors: LQ_ERR_ARG if any L < 4 or N > 2^31-1 padded sites, C <= 0 or B^2 - 24AC < 0
 * (no nematic minimum), or out == NULL; LQ_ERR_CUDA if there is no usable sm_100 device;
 * LQ_ERR_NOMEM if device memory cannot be allocated.  *out is set only on LQ_OK. */
int lq_create(int Lx, int Ly, int Lz, double A, double B, double C,
              double L1, double L2, double L3, lq_ctx **out);

/* Free the context and all device memory it owns.  NULL is allowed. */
void lq_destroy(lq_ctx *ctx);

/* Use `cuda_stream` (a cudaStream_t / CUstream passed as void*, e.g.
 * torch.cuda.current_stream().cuda_stream) for all later work.  NULL = legacy default stream. */
int lq_set_stream(lq_ctx *ctx, void *cuda_stream);

/* Geometry and anchoring: mask[N] in {LQ_SITE_LC, LQ_SITE_OBJECT};
 * anch_kind[N] in LQ_ANCH_* (NULL = none anywhere); W[N] = the coefficient W of Eq. 14 / 15
 * (NOT the Rapini-Papoular W_RP = 9 S0^2 W);
 * axis[3][N] SoA unit vectors: the preferred director n0 (kind 1) or the surface normal nu
 * (kind 2).  W and axis are read only where anch_kind != 0 and may be NULL iff anch_kind is.
 * The library classifies every site (bulk / boundary / object + 6 neighbour bits) on the GPU.
 * An anchoring term is applied at a site iff its class is boundary and its kind != 0, one term
 * per site (R9).  mask == NULL resets to "all bulk".  May be called again at any time;
 * it does not touch Q.  Errors: LQ_ERR_ARG on bad pointers / where / values > 1 in mask or > 2 in kind. */
int lq_set_sites(lq_ctx *ctx, const uint8_t *mask, const uint8_t *anch_kind,
                 const double *W, const double *axis, int where);

/* Copy the packed class/neighbour byte of every site into flags[N] (bit-exact parity gate). */
int lq_get_flags(lq_ctx *ctx, uint8_t *flags, int where);

/* Set / read the Q field, [5][N] fp64 SoA.  After lq_set_Q the FIRE velocities read as 0.
 * Values at object sites are stored and returned unchanged and never enter any result
 * (R17).  lq_get_Q before lq_set_Q: LQ_ERR_STATE. */
int lq_set_Q(lq_ctx *ctx, const double *q, int where);
int lq_get_Q(lq_ctx *ctx, double *q, int where);

/* FIRE velocities after the last lq_fire_minimize ([5][N]): the v of Algorithm 1 at the end of
 * the last step, i.e. after its rescale v <- (1-alpha) v + alpha |v| F/|F| (or v <- 0 when P <= 0); the state the
 * stop test fired on keeps its un-rescaled v.  Zeros after lq_set_Q, after lq_descent_minimize and when no step
 * was taken.  The fused sweeps apply the rescale lazily (inside the next step), so this call finishes it on a copy:
 * one force pass + one streaming pass, only when asked.  With integrator = 1 a run stopped by force_tol returns the
 * velocity already kicked with the final force. */
int lq_get_velocity(lq_ctx *ctx, double *v, int where);

/* Total free energy F = sum over simulated sites of f_bulk + f_distortion + f_anchoring
 * (PAPER.md:175): Eq. 5; Eq. 10 averaged over the forward/backward differences allowed by the
 * geometry; Eq. 14 / 15 at boundary sites.  *E is a HOST double.
 * lq_energy_terms writes (bulk, distortion, anchoring) to the host array terms[3]. */
int lq_energy(lq_ctx *ctx, double *E);
int lq_energy_terms(lq_ctx *ctx, double *terms);

/* lq_energy_terms for callers that must not allocate device memory.  lq_energy_terms keeps its per-block partial
 * sums in a buffer it cudaMalloc's on first use (and again when a larger lattice needs more).  That is a problem for a
 * host that has handed the whole GPU to a memory pool of its own (a framework's caching allocator, a service with a
 * fixed memory budget: a driver allocation may fail there or is simply forbidden), and for a latency-critical loop that
 * cannot take the device-wide synchronisation and the driver lock that cudaMalloc / cudaFree imply while other streams
 * are busy.  This entry point computes the same three numbers (bulk, distortion, anchoring; bit-identical to
 * lq_energy_terms: same kernels, same summation order) and calls no cudaMalloc, cudaFree or allocating library routine:
 * the partial sums live in a static array inside liblq.so, 1.5 MiB of every GPU that loads the library, held until the
 * process exits.
 *   - Input: the context's current Q and geometry.  Output: terms[3], caller-owned; where = LQ_DEVICE writes the three
 *     doubles on the context's stream and returns without synchronising; LQ_HOST copies them to the host and
 *     synchronises the stream before returning.
 *   - Limit: lattices of at most 65536 reduction blocks, ceil(Lx/64) * ceil(Ly/4) * ceil(Lz/8) (512^3 is exactly at the
 *     limit).  Larger: LQ_ERR_ARG, and lq_last_error names both numbers; nothing is launched.
 *   - The first call on each device looks up the array's device address (one runtime query, no allocation); make that
 *     first call before any stream capture begins.
 *   - All contexts, streams and threads share the one array per GPU.  It keeps the previous call's contents; nothing in
 *     it needs clearing, because each call overwrites every slot it later reads.  Two calls whose kernels can overlap on
 *     the GPU (different streams, or different contexts on different streams) race on it and return garbage: order them
 *     on one stream or with events.  lq_energy_terms, with its per-context buffer, has no such restriction.
 * Errors: LQ_ERR_ARG (NULL terms, bad where, lattice over the limit), LQ_ERR_STATE before lq_set_Q, LQ_ERR_CUDA. */
int lq_energy_terms_noalloc(lq_ctx *ctx, double *terms, int where);

/* Force F_a(x) = -dF/dq_a(x) in the five stored variables, [5][N], exactly 0 at
 * object sites. */
int lq_forces(lq_ctx *ctx, double *F, int where);

/* FIRE parameters (Algorithm 1).  integrator 0 = velocity Verlet as kick-drift-kick
 * (R4; the fused sweeps), 1 = plain semi-implicit Euler (R30): per step
 * v += dt F(q); P, |F|^2, |v|^2; mix; schedule; q += dt v (the step's dt, the mixed or reset v); then the new force
 * and the stop test.  Both run on the fused sweeps (the lazily applied part of a step only changes coefficients).  report_energy != 0 fills lq_fire_report.energy (one extra pass). */
typedef struct {
    double dt0, dtmax, alpha0, finc, fdec, falpha;
    int Nmin;
    int integrator;
    int report_energy;
} lq_fire_params;

/* steps = FIRE steps taken; converged = 1 iff max|F_a| < force_tol was reached (then Q is the state
 * that force was computed on); Fmax = max over simulated sites and components of |F_a|;
 * Frms = sqrt(sum F^2 / N_simulated); P = F.v of the last step; dt, alpha = schedule state after the
 * last step; energy = total energy of the final Q (0 unless report_energy);
 * launches = kernels this call launched; sweep_launches = launches of the fused force+FIRE sweep
 * kernel among them; gpu_ms = device time of the minimisation loop (CUDA events on the stream). */
typedef struct {
    long steps;
    int converged;
    double Fmax, Frms, P, dt, alpha, energy;
    long launches, sweep_launches;
    double gpu_ms;
} lq_fire_report;

/* Run FIRE from the current Q with v = 0, dt = dt0, alpha = alpha0 (state restarts every call,
 * DESIGN.md R13) until max|F_a| < force_tol or max_steps steps.  Per step: v += dt/2 F; q += dt v;
 * F = force(q); v += dt/2 F; P = F.v, |F|^2, |v|^2, max|F| over the simulated dofs;
 * v <- (1-alpha) v + alpha |v| F/|F|; P > 0: after more than Nmin such steps dt <- min(dt finc, dtmax),
 * alpha <- alpha falpha; else dt <- dt fdec, v <- 0, alpha <- alpha0 (R3).
 * The whole loop runs on the device; the host only polls a flag.  force_tol = 0 runs exactly
 * max_steps steps.  Errors: LQ_ERR_STATE before lq_set_Q; LQ_ERR_ARG on bad parameters
 * (dt0 <= 0, dtmax < dt0, alpha0 outside [0,1], finc < 1, fdec or falpha outside (0,1], Nmin < 0,
 * integrator not 0 or 1, max_steps < 0, NULL pointers). */
int lq_fire_minimize(lq_ctx *ctx, long max_steps, double force_tol,
                     const lq_fire_params *params, lq_fire_report *out);

/* Uniform external magnetic / electric fields, Eq. 13:
 *     f_external = -(1/3) chi H_i Q_ij H_j - (1/3) eps E_i Q_ij E_j        at every simulated site,
 * chi = mu0 Delta-chi and eps = eps0 Delta-eps in the context's nondimensional units (positive values favour
 * alignment of the director with the field).  H, E: host double[3] (NULL = zero vector).  The term enters
 * lq_energy (reported inside the bulk term of lq_energy_terms), lq_forces and every minimiser; it costs no extra
 * instruction in the kernels (a constant folded into existing FMAs).  Calling it again replaces the fields;
 * all-zero arguments switch the term off.  Errors: LQ_ERR_ARG on non-finite values. */
int lq_set_field(lq_ctx *ctx, const double *H, double chi, const double *E, double eps);

/* Chiral distortion constant L4 of Eq. 10: adds
 *     L4/2 eps_lik Q_lj dQ_ij/dx_k      (in the uniaxial limit L4 = -(8 / 9 S^2) q0 K2)
 * to the distortion energy of every simulated site, with the same averaged one-sided differences as the other terms
 * (the term is linear in the derivative, so the average over the allowed sign combinations is the expression on the
 * mean differences).  L4 != 0 routes every minimiser through the 19-point sweeps (like L2, L3 != 0), whose
 * constant-weight stencil gains L4 eps_aik C_k Q_ib (C_k = centred difference).
 * L4 = 0 switches the term off.  Errors: LQ_ERR_ARG on a non-finite value. */
int lq_set_chiral(lq_ctx *ctx, double L4);

/* Cubic distortion constant L6 of Eq. 10: adds L6/2 Q_lk dQ_ij/dx_l dQ_ij/dx_k (in the uniaxial
 * limit L6 = (4 / 27 S^3)(K3 - K1): it separates bend from splay).  Discretised like L1..L3: same-axis
 * products average to the mean of the squared one-sided differences, different-axis products to products of the
 * mean differences; the weight Q_lk is the site's own tensor.  Routed like lq_set_chiral (19-point sweeps with the
 * term compiled in, on 32 x 8 tiles so that they fit the register budget without spilling).  Errors as
 * lq_set_chiral. */
int lq_set_cubic(lq_ctx *ctx, double L6);

/* Other first-order minimisers on the same force.  The paper compares FIRE with gradient
 * descent and offers Nesterov's accelerated gradient as its second minimiser
 * without printing either update; the fixed-step textbook forms are used
 * (R23, R24):
 *     LQ_MIN_GD:        y_k = q_k
 *     LQ_MIN_NESTEROV:  y_k = q_k + mu (q_k - q_{k-1}),  q_{-1} = q_0
 *     q_{k+1} = y_k + eta F(y_k) on simulated sites; object sites never move.
 * One kernel launch per step.  The stop test max|F_a(y_k)| < force_tol uses the force the step evaluates and
 * the step's update is still applied, so steps = updates applied (force_tol = 0: exactly max_steps).
 * The report reuses lq_fire_report: Fmax, Frms of F(y_k) of the last step; P = 0; dt = eta; alpha = mu.
 * lq_get_velocity returns zeros afterwards (these minimisers carry no velocity).
 * Errors: LQ_ERR_STATE before lq_set_Q; LQ_ERR_ARG on eta <= 0, mu outside [0, 1), unknown method,
 * max_steps < 0, NULL pointers. */
enum { LQ_MIN_GD = 0, LQ_MIN_NESTEROV = 1 };
typedef struct {
    double eta;          /* step size */
    double mu;           /* momentum of LQ_MIN_NESTEROV (ignored by LQ_MIN_GD) */
    int report_energy;
} lq_descent_params;
int lq_descent_minimize(lq_ctx *ctx, int method, long max_steps, double force_tol,
                        const lq_descent_params *params, lq_fire_report *out);

/* Per-site analysis of the current Q: "The nematic director can be recovered as the eigenvector
 * corresponding to the largest eigenvalue of Q, which equals S" (Eq. 2); defects are "regions where
 * the largest eigenvalue of Q falls below some threshold".  Outputs are dense (unpadded) arrays in
 * lattice order s = x + Lx (y + Ly z), each may be NULL: S [N]; director [3][N] SoA, unit length, the component of
 * largest magnitude positive (first such on ties; the director is headless); defect [N] bytes, 1 where
 * S < S_threshold; *n_defect (host long) = number of such sites.  Object sites get S = 0, director = 0, defect = 0.
 * Where the largest eigenvalue is degenerate the director is any unit vector of its eigenspace.
 * One streaming kernel launch.  Errors: LQ_ERR_STATE before lq_set_Q, LQ_ERR_ARG on a bad `where`. */
int lq_analyze(lq_ctx *ctx, double S_threshold, double *S, double *director, uint8_t *defect, long *n_defect,
               int where);

/* ---- Domain decomposition into z-slabs.  The paper uses "a standard spatial decomposition of the total
 * number of lattice sites into rectilinear sub-regions"; "each processing unit is assigned to one of these subregions"
 * and also keeps the state of the halo sites, which are communicated every simulation step (sec.
 * III.B; the weak-scaling workload of Fig. 4).  The paper does not spell out the reduction of the
 * minimiser's scalars over the units; FIRE needs one (P, |F|^2, |v|^2, max|F| are global), so it is part of the
 * protocol here.  Here: slabs along z.
 *
 * lq_create_slab makes a sub-domain context for the planes [z0, z0 + nz) of a global Lx x Ly x Lz lattice (nz >= 4).
 * It behaves like any context on LOCAL arrays of nz planes (lq_set_Q, lq_get_Q, lq_get_flags, lq_forces, lq_energy,
 * lq_analyze: the slab's own sites), with these differences: nothing wraps in z -- the two ghost planes on either
 * side hold the neighbour slabs' boundary planes and are filled by a halo exchange, which must follow every
 * lq_set_Q before lq_energy / lq_forces / a FIRE run; geometry comes through lq_set_sites_ext; FIRE runs through
 * lq_slabs_fire_minimize (same process, same GPU) or lq_fire_begin / step_local / step_commit / end (one rank per
 * GPU); lq_fire_minimize, lq_descent_minimize and fire_path 1 return LQ_ERR_STATE. */
int lq_create_slab(int Lx, int Ly, int Lz_global, int z0, int nz, double A, double B, double C,
                   double L1, double L2, double L3, lq_ctx **out);

/* Geometry of a sub-domain: like lq_set_sites, but every array covers the planes z0-3 .. z0+nz+2 of the global
 * lattice (periodic wrap in z), i.e. (nz + 6) * Ly * Lx sites ([3][...] for axis): the 3-plane margin makes the
 * classification of the slab's two ghost planes, and with it every stencil weight near a face, identical to the
 * undivided lattice's (bit-exact flags: lq_get_flags returns the slab's nz planes). */
int lq_set_sites_ext(lq_ctx *ctx, const uint8_t *mask_ext, const uint8_t *kind_ext, const double *W_ext,
                     const double *axis_ext, int where);

/* Halo packages.  what = LQ_HALO_Q: the Q field (after lq_set_Q); LQ_HALO_STATE: the FIRE state after a step
 * (q, v, and the stored force on the stored-force path).  face 0 = low z, 1 = high z.  lq_halo_export packs the
 * slab's own two boundary planes of that face (z = 0, 1 or nz-2, nz-1; whole padded planes, 5 components per field)
 * into buf (lq_halo_bytes bytes); lq_halo_import writes a package into the two ghost planes of that face
 * (z = -2, -1 or nz, nz+1).  A slab's low-face ghosts take its lower neighbour's HIGH-face export and vice versa
 * (periodic in the slab index).  lq_slabs_exchange does this for a whole same-process group with device-to-device
 * copies and returns when they have completed. */
enum { LQ_HALO_Q = 0, LQ_HALO_STATE = 1 };
int lq_halo_bytes(lq_ctx *ctx, int what, size_t *bytes);
int lq_halo_export(lq_ctx *ctx, int what, int face, void *buf, int where);
int lq_halo_import(lq_ctx *ctx, int what, int face, const void *buf, int where);
int lq_slabs_exchange(lq_ctx **slabs, int n, int what);

/* FIRE over a same-process group of slabs that tile [0, Lz) in z order, all on one GPU and one stream: per step one
 * fused sweep per slab (schedule update deferred), one reduction kernel over all slabs' per-CTA partials in a fixed
 * order (the "all-reduce" of (P, |F|^2, |v|^2, max|F|)), one kernel that writes the same schedule update into every
 * slab's device scalars, and device-to-device halo copies.  The report is that of the whole lattice. */
int lq_slabs_fire_minimize(lq_ctx **slabs, int n, long max_steps, double force_tol,
                           const lq_fire_params *params, lq_fire_report *out);

/* The same step in transport-agnostic pieces, for one rank per GPU.  After the initial LQ_HALO_Q exchange:
 *     lq_fire_begin(ctx, ...)
 *     repeat: lq_fire_step_local(ctx)            the fused sweep of this slab (schedule update deferred)
 *             exchange LQ_HALO_STATE packages with both neighbours
 *             lq_fire_step_finish(ctx, tot6, where, &again)   the fix-up launch where the path has one (stored force
 *                                                + objects: it evaluates forces on q' across the faces), then this
 *                                                slab's row (P, |F|^2, |v|^2, max|F|, and for the first sweep
 *                                                |F(q_0)|^2, max|F(q_0)|), to a device or host buffer
 *             all-gather the rows;  lq_fire_step_commit(ctx, rows, nrank): rows combined in rank order -> schedule
 *             if again: exchange LQ_HALO_STATE once more (the fix-up changed v and F on the boundary planes)
 *             every so often lq_fire_peek(ctx, report) (synchronises) to test `converged`
 *     lq_fire_end(ctx, report)                   fixes the live buffer; Frms uses the slab's own site count
 * The number of sweeps to enqueue is max(max_steps, 1), or max_steps + 1 on the stored-force path or with
 * integrator = 1; lq_get_info(ctx, "fire_sweeps_total") returns it after lq_fire_begin.  Either every slab of a lattice
 * gets geometry (lq_set_sites_ext) or none does.
 * Stream order.  With where = LQ_DEVICE, lq_halo_export, lq_halo_import, lq_fire_step_finish and lq_fire_step_commit
 * only ENQUEUE work on the context's stream (lq_set_stream) and return: the caller's device buffer is written / read
 * when the stream gets there, not when the call returns.  Anything that touches such a buffer on another stream (a
 * communication library, the caller's own kernels) must be ordered against the context's stream with events or by
 * running on that stream, and the buffer must stay allocated until the enqueued work has run.  With where = LQ_HOST the
 * same calls synchronise the context's stream before returning, so the host buffer is complete (or free to reuse) on
 * return.  lq_fire_step_local and lq_fire_begin always only enqueue; lq_fire_peek and lq_fire_end synchronise. */
int lq_fire_begin(lq_ctx *ctx, long max_steps, double force_tol, const lq_fire_params *params);
int lq_fire_step_local(lq_ctx *ctx);
int lq_fire_step_finish(lq_ctx *ctx, double *tot6, int where, int *exchange_again);
int lq_fire_step_commit(lq_ctx *ctx, const double *rows, int nrank, int where);
int lq_fire_peek(lq_ctx *ctx, lq_fire_report *out);
int lq_fire_end(lq_ctx *ctx, lq_fire_report *out);

/* S0 of Eq. 7 for the context's A, B, C (host double). */
int lq_get_S0(lq_ctx *ctx, double *S0);

/* Tuning / introspection, not part of the method.  Keys:
 *   "fire_path" (set): 0 = fused one-launch-per-step sweep (default; one-constant: force recomputed,
 *                      state (q, v); L2/L3 != 0: force stored, state (q, v, F)), 1 = unfused four-kernel
 *                      path, 2 = fused sweep with the force stored (any constants).
 *                      lq_descent_minimize: 0 = TMA sweep over the constant-weight sites + list kernel for the
 *                      rest, 1 = general kernel on every site
 *   "resident" (set):  1 (default) = one-constant lattices small enough to live on chip (bricks of <= 512 sites on
 *                      <= one CTA per SM, about 75 000 sites on a B200) run lq_fire_minimize (integrator 0,
 *                      fire_path 0) as ONE cooperative launch with q, v, F in registers / shared memory and one grid
 *                      barrier per step; report.sweep_launches is then 1.  0 = always the streaming sweeps
 *   "rc_chunks" (set): recompute sweep: 0 = z-chunks per tile column chosen by the makespan model (default),
 *                      n > 0 = n equal chunks per column (clamped to chunks of 4 .. 126 planes)
 *   "sweep_bytes_per_site" (get): algorithmic HBM bytes one sweep moves per site
 *   "n_simulated" (get), "n_boundary" (get), "n_object" (get)
 *   "has_fixup" (get): 1 if a FIRE step on this context is a sweep plus a fix-up launch (stored force + objects)
 *   "stored_force" (get): 1 if the fused FIRE sweep of this context keeps the force in memory (state (q, v, F): three
 *                      constants, L4 / L6, or fire_path 2), 0 if it recomputes it (state (q, v))
 *   "fire_sweeps_total" (get): between lq_fire_begin and lq_fire_end: the number of lq_fire_step_local rounds a full run
 *                      of max_steps steps takes (see the step-wise protocol above); LQ_ERR_STATE otherwise
 *   "fp64_fma_tflops" (get): runs a register-only fp64 FMA microbenchmark on the context's device and stream (a few
 *                      milliseconds) and returns the measured TFLOP/s: the ALU roof next to the HBM one
 * Unknown key: LQ_ERR_ARG. */
int lq_set_option(lq_ctx *ctx, const char *key, double value);
int lq_get_info(lq_ctx *ctx, const char *key, double *value);

/* Message for the last error on this context ("" if none); valid until the next call. */
const char *lq_last_error(lq_ctx *ctx);

/* Library version string, e.g. "lq 0.1 sm_100a". */
const char *lq_version(void);

#ifdef __cplusplus
}
#endif
#endif /* LQ_H */

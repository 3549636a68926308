/*
 * lq_oracle.c — CPU ORACLE for the Landau-de Gennes / FIRE hot path.
 *
 * THIS FILE IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  It is a plain, slow,
 * fp64 restatement of what arXiv:1911.07045 (Sussman & Beller, "openQmin")
 * says the method computes.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may call it.  It shares no
 * code, header, table or helper with paper_1911_07045_b200/csrc (the CUDA
 * path), and neither includes the other.
 *
 * Citations are "PAPER.md:<line>" = /root/reference/PAPER.md plus the section
 * or equation the line falls in.  "DESIGN.md Rn" = a reading of a silent /
 * garbled passage, listed in DESIGN.md section 3.
 *
 * Two separately written evaluations of the same discretised free energy:
 *   variant 0  "literal"   : per site, enumerate every allowed combination of
 *                            forward/backward differences,
 *                            evaluate Eq. 10 on full 3x3 tensors with index
 *                            loops, average; gradient by the product rule on
 *                            those same loops, scattered to the 7 sites the
 *                            site energy touches.  Serial.  The arbiter.
 *   variant 1  "factorised": uses the algebraic identity that the average of
 *                            a quadratic form over a product set of signs is
 *                            (mean of squares) for same-axis terms and
 *                            (product of mean differences) for mixed terms;
 *                            scatter gradient; OpenMP over z-planes with a
 *                            3-colouring.  Checked against variant 0 in
 *                            tests/test_oracle_pins.py; used on large configs
 *                            and for the timed CPU baseline.
 *
 * Pins (tests/test_oracle_pins.py, -m "not gpu"): S0/f0 closed forms (Eq. 6-8),
 * zero elastic force on uniform fields, force == -central finite difference of
 * the total energy on tiny masked lattices, plane-wave/checkerboard response,
 * L2 == L3 on periodic object-free lattices, anchoring closed forms
 * (W_RP = 9 S0^2 W), translation / rotation invariance, FIRE
 * schedule hand trace, classification counts.  Later additions and their pins:
 * gradient descent / Nesterov (lqo_descent; tests/test_oracle_descent.py: Eq. 6
 * scalar recurrence, plane-wave linear recurrences, descent lemma); the external
 * field term of Eq. 13 (tests/test_field.py: the uniaxial limit printed under
 * Eq. 13, constant force by hand, finite differences, alignment with H); the
 * chiral L4 term (tests/test_chiral.py: hand-derived helix energy, the printed
 * L4 <-> q0 K2 map, preferred pitch) and the cubic L6 term (tests/test_cubic.py:
 * the printed L <-> K map on twist / splay / bend fields) of Eq. 10; the
 * director / S / defect analysis lives in lq_oracle.py (numpy.linalg.eigh;
 * tests/test_analyze.py: Eq. 2 and Eq. 3 round trips).
 * The L2-vs-L3 split of Eq. 10 next to objects (tests/test_oracle_pins.py: hand-
 * evaluated ramp fields where only L2 carries the cross product, and the wall
 * surface sum that E(L2) - E(L3) reduces to by discrete summation by parts).
 * Parity UNPINNED: the FIRE / GD / Nesterov trajectories on the full-size
 * configs 3 and 5 (no published numbers) -- GPU-vs-oracle only.
 *
 * Layout: fields are SoA, q[c*N + s], c in (xx,xy,xz,yy,yz),
 * s = x + Lx*(y + Ly*z); Qzz = -Qxx-Qyy.  Index arithmetic is periodic in all
 * three directions; walls are layers of object sites (R14).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef struct {
    int Lx, Ly, Lz;
    double A, B, C;          /* bulk constants, Eq. 5            */
    double L1, L2, L3;       /* distortion constants, Eq. 10    */
    const uint8_t *mask;     /* [N] 0 = liquid crystal, 1 = object; NULL = all 0 */
    const uint8_t *kind;     /* [N] 0 none, 1 oriented (Eq.14), 2 degenerate planar (Eq.15); NULL = none */
    const double *W;         /* [N] anchoring strength of Eq. 14/15; NULL if kind NULL */
    const double *axis;      /* [3][N] unit vector n0 (kind 1) or nu (kind 2)  */
    /* external fields, Eq. 13: uniform H and E; chi = mu0 Delta-chi, eps = eps0 Delta-eps */
    double H[3], chi, E[3], eps;
    double L4;               /* chiral distortion constant of Eq. 10 */
    double L6;               /* cubic distortion constant of Eq. 10 */
} lqo_problem;

typedef struct { double dt0, dtmax, alpha0, finc, fdec, falpha; int Nmin; int integrator; } lqo_fire_params;
typedef struct { long steps; int converged; double Fmax, Frms, P, dt, alpha, energy; } lqo_fire_report;

/* ------------------------------------------------------------------ basics */

static inline int wrapi(int i, int L) { return i < 0 ? i + L : (i >= L ? i - L : i); }
static inline long site_of(const lqo_problem *p, int x, int y, int z)
{ return (long)x + (long)p->Lx * ((long)y + (long)p->Ly * (long)z); }
static inline int is_sim(const lqo_problem *p, long s) { return p->mask == NULL || p->mask[s] == 0; }

/* neighbour of (x,y,z) along axis k (0,1,2) with sign sg (+1/-1), periodic */
static inline long nbr_of(const lqo_problem *p, int x, int y, int z, int k, int sg)
{
    if (k == 0) x = wrapi(x + sg, p->Lx);
    else if (k == 1) y = wrapi(y + sg, p->Ly);
    else z = wrapi(z + sg, p->Lz);
    return site_of(p, x, y, z);
}

/* full symmetric traceless 3x3 tensor from the 5 stored numbers */
static inline void load_Q(const double *q, long N, long s, double Q[3][3])
{
    double xx = q[s], xy = q[N + s], xz = q[2 * N + s], yy = q[3 * N + s], yz = q[4 * N + s];
    Q[0][0] = xx; Q[0][1] = xy; Q[0][2] = xz;
    Q[1][0] = xy; Q[1][1] = yy; Q[1][2] = yz;
    Q[2][0] = xz; Q[2][1] = yz; Q[2][2] = -xx - yy;
}

/* chain rule from the 9 tensor-entry derivatives G_ab = dE/dQ_ab (entries
 * treated as independent) to the 5 stored variables:  Qyx=Qxy, Qzx=Qxz,
 * Qzy=Qyz, Qzz=-Qxx-Qyy ("explicitly differentiating ...
 * with respect to each q_i"). */
static inline void G_to_5(const double G[3][3], double g5[5])
{
    g5[0] = G[0][0] - G[2][2];
    g5[1] = G[0][1] + G[1][0];
    g5[2] = G[0][2] + G[2][0];
    g5[3] = G[1][1] - G[2][2];
    g5[4] = G[1][2] + G[2][1];
}

/* Eq. 7: S0 = (-B + sqrt(B^2 - 24 A C)) / (6 C) */
double lqo_S0(double A, double B, double C) { return (-B + sqrt(B * B - 24.0 * A * C)) / (6.0 * C); }
/* amplitude of the uniaxial tensor Q = q0 (nn - I/3):  q0 = (3/2) S0  (Eq. 3) */
double lqo_q0(double A, double B, double C) { return 1.5 * lqo_S0(A, B, C); }

int lqo_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
void lqo_set_num_threads(int n)
{
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

/* ---------------------------------------------------------- classification
 * integer type per site: bulk / boundary / inside-object.
 * DESIGN.md R8: boundary = simulated site with at least one of its 6 face
 * neighbours (periodic wrap) an object site.  Packed byte:
 *   bits 0-1 class (0 bulk, 1 boundary, 2 object)
 *   bit 2 (+x) 3 (-x) 4 (+y) 5 (-y) 6 (+z) 7 (-z): that neighbour is simulated
 *   (set the same way at object sites).                                       */
void lqo_classify(const lqo_problem *p, uint8_t *flags)
{
    for (int z = 0; z < p->Lz; ++z)
        for (int y = 0; y < p->Ly; ++y)
            for (int x = 0; x < p->Lx; ++x) {
                long s = site_of(p, x, y, z);
                unsigned f = 0;
                int any_obj = 0;
                for (int k = 0; k < 3; ++k)
                    for (int sg = +1; sg >= -1; sg -= 2) {
                        long t = nbr_of(p, x, y, z, k, sg);
                        int bit = 2 + 2 * k + (sg < 0 ? 1 : 0);
                        if (is_sim(p, t)) f |= (1u << bit);
                        else any_obj = 1;
                    }
                unsigned cls = !is_sim(p, s) ? 2u : (any_obj ? 1u : 0u);
                flags[s] = (uint8_t)(f | cls);
            }
}

/* ------------------------------------------------------- local energy terms */

/* Eq. 5 on the full tensor, traces by index loops */
static double bulk_energy(const lqo_problem *p, const double Q[3][3])
{
    double tr2 = 0.0, tr3 = 0.0;
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j) {
            tr2 += Q[i][j] * Q[j][i];
            for (int k = 0; k < 3; ++k) tr3 += Q[i][j] * Q[j][k] * Q[k][i];
        }
    return 0.5 * p->A * tr2 + p->B / 3.0 * tr3 + 0.25 * p->C * tr2 * tr2;
}

/* Eq. 13: f_external = -(1/3) chi H_i Q_ij H_j - (1/3) eps E_i Q_ij E_j */
static double field_energy(const lqo_problem *p, const double Q[3][3])
{
    double e = 0.0;
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j)
            e -= (p->chi * p->H[i] * Q[i][j] * p->H[j] + p->eps * p->E[i] * Q[i][j] * p->E[j]) / 3.0;
    return e;
}
/* d(f_external)/dQ_ab, entries independent: linear in Q, so a constant tensor */
static void field_grad_add(const lqo_problem *p, double G[3][3])
{
    for (int a = 0; a < 3; ++a)
        for (int b = 0; b < 3; ++b)
            G[a][b] -= (p->chi * p->H[a] * p->H[b] + p->eps * p->E[a] * p->E[b]) / 3.0;
}

/* d(bulk)/dQ_ab with entries independent:
 *   d tr(Q^2)/dQ_ab = 2 Q_ba ; d tr(Q^3)/dQ_ab = 3 (Q^2)_ba                    */
static void bulk_grad(const lqo_problem *p, const double Q[3][3], double G[3][3])
{
    double tr2 = 0.0, Q2[3][3];
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j) {
            tr2 += Q[i][j] * Q[j][i];
            double a = 0.0;
            for (int k = 0; k < 3; ++k) a += Q[i][k] * Q[k][j];
            Q2[i][j] = a;
        }
    for (int a = 0; a < 3; ++a)
        for (int b = 0; b < 3; ++b)
            G[a][b] = p->A * Q[b][a] + p->B * Q2[b][a] + p->C * tr2 * Q[b][a];
}

/* Anchoring energy of one boundary site (R9: one term per boundary
 * site, and only there: `boundary` = the site's class is boundary; kind set on a bulk site adds nothing).  kind 1: Eq. 14, Q0 = (3/2) S0 (n n - I/3).
 * kind 2: Eq. 15 with the garbled projection read as
 * Qt_perp = P Qt P (R2), Qt = Q + (S0/2) I, P = I - nu nu.
 * Returns the energy; if G != NULL also d/dQ_ab.                              */
static double anchoring(const lqo_problem *p, long N, long s, int boundary, const double Q[3][3], double G[3][3])
{
    if (G) memset(G, 0, 9 * sizeof(double));
    /* SURVEY 8(c) O5 / DESIGN.md R9: a term only where class == boundary and kind != 0 */
    if (!boundary || p->kind == NULL || p->kind[s] == 0) return 0.0;
    const double S0 = lqo_S0(p->A, p->B, p->C);
    const double W = p->W[s];
    const double n[3] = { p->axis[s], p->axis[N + s], p->axis[2 * N + s] };
    double e = 0.0;
    if (p->kind[s] == 1) {
        for (int i = 0; i < 3; ++i)
            for (int j = 0; j < 3; ++j) {
                double Q0 = 1.5 * S0 * (n[i] * n[j] - (i == j ? 1.0 / 3.0 : 0.0));
                double d = Q[i][j] - Q0;
                e += W * d * d;
                if (G) G[i][j] = 2.0 * W * d;
            }
    } else if (p->kind[s] == 2) {
        double Qt[3][3], P[3][3], PQ[3][3], M[3][3];
        for (int i = 0; i < 3; ++i)
            for (int j = 0; j < 3; ++j) {
                Qt[i][j] = Q[i][j] + (i == j ? 0.5 * S0 : 0.0);
                P[i][j] = (i == j ? 1.0 : 0.0) - n[i] * n[j];
            }
        for (int i = 0; i < 3; ++i)
            for (int j = 0; j < 3; ++j) {
                double a = 0.0;
                for (int k = 0; k < 3; ++k) a += P[i][k] * Qt[k][j];
                PQ[i][j] = a;
            }
        for (int i = 0; i < 3; ++i)
            for (int j = 0; j < 3; ++j) {
                double a = 0.0;
                for (int k = 0; k < 3; ++k) a += PQ[i][k] * P[k][j];
                M[i][j] = Qt[i][j] - a;   /* Qt - P Qt P */
                e += W * M[i][j] * M[i][j];
            }
        if (G) {
            /* e = W sum_ij M_ij^2, M = Qt - P Qt P is linear in Q:
             * de/dQ_ab = 2 W sum_ij M_ij (d_ia d_jb - P_ia P_bj) = 2 W (M - P M P)_ab
             * (P symmetric).  Written out literally, no use of projector identities. */
            double PM[3][3];
            for (int i = 0; i < 3; ++i)
                for (int j = 0; j < 3; ++j) {
                    double a = 0.0;
                    for (int k = 0; k < 3; ++k) a += P[i][k] * M[k][j];
                    PM[i][j] = a;
                }
            for (int a = 0; a < 3; ++a)
                for (int b = 0; b < 3; ++b) {
                    double pmp = 0.0;
                    for (int k = 0; k < 3; ++k) pmp += PM[a][k] * P[k][b];
                    G[a][b] = 2.0 * W * (M[a][b] - pmp);
                }
        }
    }
    return e;
}

/* boundary class (R8): a simulated site with at least one of its 6 face
 * neighbours (periodic wrap) an object site */
static int is_boundary_site(const lqo_problem *p, int x, int y, int z)
{
    if (!is_sim(p, site_of(p, x, y, z))) return 0;
    for (int k = 0; k < 3; ++k)
        for (int sg = +1; sg >= -1; sg -= 2)
            if (!is_sim(p, nbr_of(p, x, y, z, k, sg))) return 1;
    return 0;
}

/* allowed finite-difference signs per axis at a simulated site.
 * DESIGN.md R6: if neither neighbour along an axis is simulated the derivative
 * along that axis is taken as 0 (a single "sign 0" option).                   */
static void allowed_signs(const lqo_problem *p, int x, int y, int z, int nopt[3], int opt[3][2])
{
    for (int k = 0; k < 3; ++k) {
        nopt[k] = 0;
        if (is_sim(p, nbr_of(p, x, y, z, k, +1))) opt[k][nopt[k]++] = +1;
        if (is_sim(p, nbr_of(p, x, y, z, k, -1))) opt[k][nopt[k]++] = -1;
        if (nopt[k] == 0) { opt[k][0] = 0; nopt[k] = 1; }
    }
}

/* Levi-Civita symbol */
static inline double eps3(int i, int j, int k) { return (double)((i - j) * (j - k) * (k - i)) / 2.0; }

/* Eq. 10, all five terms, for one choice of difference tensors
 * D[k][i][j] ~ dQ_ij/dx_k and the site's own tensor Q (the chiral term
 * L4/2 eps_lik Q_lj dQ_ij/dx_k carries an undifferentiated Q); index loops
 * exactly as printed.  If gD != NULL it receives d f / d D[k][i][j] and gQ
 * d f / d Q[l][j] (entries independent) by the product rule term by term.     */
static double f_distortion(const lqo_problem *p, const double Q[3][3], const double D[3][3][3],
                           double gD[3][3][3], double gQ[3][3])
{
    double f = 0.0;
    if (gD) { memset(gD, 0, 27 * sizeof(double)); memset(gQ, 0, 9 * sizeof(double)); }
    if (p->L6 != 0.0)
        for (int l = 0; l < 3; ++l)
            for (int k = 0; k < 3; ++k)
                for (int i = 0; i < 3; ++i)
                    for (int j = 0; j < 3; ++j) {
                        /* L6/2 Q_lk dQij/dxl dQij/dxk */
                        f += 0.5 * p->L6 * Q[l][k] * D[l][i][j] * D[k][i][j];
                        if (gD) {
                            gD[l][i][j] += 0.5 * p->L6 * Q[l][k] * D[k][i][j];
                            gD[k][i][j] += 0.5 * p->L6 * Q[l][k] * D[l][i][j];
                            gQ[l][k] += 0.5 * p->L6 * D[l][i][j] * D[k][i][j];
                        }
                    }
    if (p->L4 != 0.0)
        for (int l = 0; l < 3; ++l)
            for (int i = 0; i < 3; ++i)
                for (int k = 0; k < 3; ++k) {
                    const double e = eps3(l, i, k);
                    if (e == 0.0) continue;
                    for (int j = 0; j < 3; ++j) {
                        /* L4/2 eps_lik Q_lj dQij/dxk */
                        f += 0.5 * p->L4 * e * Q[l][j] * D[k][i][j];
                        if (gD) {
                            gD[k][i][j] += 0.5 * p->L4 * e * Q[l][j];
                            gQ[l][j] += 0.5 * p->L4 * e * D[k][i][j];
                        }
                    }
                }
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j)
            for (int k = 0; k < 3; ++k) {
                /* L1/2 dQij/dxk dQij/dxk */
                f += 0.5 * p->L1 * D[k][i][j] * D[k][i][j];
                /* L2/2 dQij/dxj dQik/dxk */
                f += 0.5 * p->L2 * D[j][i][j] * D[k][i][k];
                /* L3/2 dQik/dxj dQij/dxk */
                f += 0.5 * p->L3 * D[j][i][k] * D[k][i][j];
                if (gD) {
                    gD[k][i][j] += p->L1 * D[k][i][j];
                    gD[j][i][j] += 0.5 * p->L2 * D[k][i][k];
                    gD[k][i][k] += 0.5 * p->L2 * D[j][i][j];
                    gD[j][i][k] += 0.5 * p->L3 * D[k][i][j];
                    gD[k][i][j] += 0.5 * p->L3 * D[j][i][k];
                }
            }
    return f;
}

/* --------------------------------------------------- variant 0: literal site
 * Energy of one site = bulk + (mean over allowed sign combinations of Eq. 10)
 * + anchoring.  terms[0..2] += (bulk, distortion, anchor).
 * If g != NULL: g[slot][5] receives d(site energy)/d(q of slot's site),
 * slot 0 = the site itself, slot 1+2k = neighbour +k, slot 2+2k = neighbour -k. */
static double site_literal(const lqo_problem *p, const double *q, int x, int y, int z,
                           double terms[3], double g[7][5])
{
    const long N = (long)p->Lx * p->Ly * p->Lz;
    const long s = site_of(p, x, y, z);
    if (g) memset(g, 0, 35 * sizeof(double));
    if (!is_sim(p, s)) return 0.0;

    double Q[3][3], Qn[3][2][3][3];
    load_Q(q, N, s, Q);
    for (int k = 0; k < 3; ++k) {
        load_Q(q, N, nbr_of(p, x, y, z, k, +1), Qn[k][0]);
        load_Q(q, N, nbr_of(p, x, y, z, k, -1), Qn[k][1]);
    }
    double G9[7][3][3];
    memset(G9, 0, sizeof(G9));

    double eb = bulk_energy(p, Q) + field_energy(p, Q);      /* the "bulk" slot carries Eq. 13 too */
    if (g) { bulk_grad(p, Q, G9[0]); field_grad_add(p, G9[0]); }

    int nopt[3], opt[3][2];
    allowed_signs(p, x, y, z, nopt, opt);
    const int ncombo = nopt[0] * nopt[1] * nopt[2];
    double ed = 0.0;
    for (int a = 0; a < nopt[0]; ++a)
        for (int b = 0; b < nopt[1]; ++b)
            for (int c = 0; c < nopt[2]; ++c) {
                const int sg[3] = { opt[0][a], opt[1][b], opt[2][c] };
                double D[3][3][3], gD[3][3][3], gQ[3][3];
                for (int k = 0; k < 3; ++k)
                    for (int i = 0; i < 3; ++i)
                        for (int j = 0; j < 3; ++j) {
                            /* Eq. 16: forward Q(x+k)-Q(x), backward Q(x)-Q(x-k) */
                            if (sg[k] > 0) D[k][i][j] = Qn[k][0][i][j] - Q[i][j];
                            else if (sg[k] < 0) D[k][i][j] = Q[i][j] - Qn[k][1][i][j];
                            else D[k][i][j] = 0.0;
                        }
                ed += f_distortion(p, Q, D, g ? gD : NULL, gQ) / ncombo;
                if (g)
                    for (int i = 0; i < 3; ++i)
                        for (int j = 0; j < 3; ++j) G9[0][i][j] += gQ[i][j] / ncombo;
                if (g)
                    for (int k = 0; k < 3; ++k) {
                        if (sg[k] == 0) continue;
                        const int slot = 1 + 2 * k + (sg[k] < 0 ? 1 : 0);
                        for (int i = 0; i < 3; ++i)
                            for (int j = 0; j < 3; ++j) {
                                /* forward: dD/dQ(x+k)=+1, dD/dQ(x)=-1; backward: dD/dQ(x)=+1, dD/dQ(x-k)=-1 */
                                const double w = gD[k][i][j] / ncombo;
                                if (sg[k] > 0) { G9[slot][i][j] += w; G9[0][i][j] -= w; }
                                else           { G9[0][i][j] += w; G9[slot][i][j] -= w; }
                            }
                    }
            }

    double Ga[3][3];
    double ea = anchoring(p, N, s, is_boundary_site(p, x, y, z), Q, g ? Ga : NULL);
    if (g)
        for (int i = 0; i < 3; ++i)
            for (int j = 0; j < 3; ++j) G9[0][i][j] += Ga[i][j];

    if (g) for (int t = 0; t < 7; ++t) G_to_5(G9[t], g[t]);
    if (terms) { terms[0] += eb; terms[1] += ed; terms[2] += ea; }
    return eb + ed + ea;
}

/* ------------------------------------------------ variant 1: factorised site
 * Same site energy, using: for a quadratic form averaged over a product set of
 * signs, same-axis products average to (1/|A_k|) sum_s D^s_k a D^s_k b and
 * different-axis products to Dbar_j a * Dbar_k b with Dbar_k the mean of the
 * allowed one-sided differences (R5/R7).  Separately written from
 * site_literal; agreement is a test, not an assumption.                       */
static double site_factorised(const lqo_problem *p, const double *q, int x, int y, int z,
                              double terms[3], double g[7][5])
{
    const long N = (long)p->Lx * p->Ly * p->Lz;
    const long s = site_of(p, x, y, z);
    if (g) memset(g, 0, 35 * sizeof(double));
    if (!is_sim(p, s)) return 0.0;

    double Q[3][3];
    load_Q(q, N, s, Q);
    double Ds[3][2][3][3];   /* one-sided differences: [axis][0 fwd,1 bwd] */
    int ok[3][2], cnt[3];
    double Dbar[3][3][3];
    for (int k = 0; k < 3; ++k) {
        cnt[k] = 0;
        for (int d = 0; d < 2; ++d) {
            const int sgn = d == 0 ? +1 : -1;
            const long t = nbr_of(p, x, y, z, k, sgn);
            ok[k][d] = is_sim(p, t);
            if (ok[k][d]) {
                double Qt[3][3];
                load_Q(q, N, t, Qt);
                for (int i = 0; i < 3; ++i)
                    for (int j = 0; j < 3; ++j)
                        Ds[k][d][i][j] = sgn > 0 ? Qt[i][j] - Q[i][j] : Q[i][j] - Qt[i][j];
                cnt[k]++;
            } else
                memset(Ds[k][d], 0, 9 * sizeof(double));
        }
        for (int i = 0; i < 3; ++i)
            for (int j = 0; j < 3; ++j)
                Dbar[k][i][j] = cnt[k] ? (Ds[k][0][i][j] + Ds[k][1][i][j]) / cnt[k] : 0.0;
    }

    double gDs[3][2][3][3], gDbar[3][3][3];
    memset(gDs, 0, sizeof(gDs));
    memset(gDbar, 0, sizeof(gDbar));
    double ed = 0.0;
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j)
            for (int k = 0; k < 3; ++k) {
                /* L1 term: always same axis k twice */
                for (int d = 0; d < 2; ++d)
                    if (ok[k][d]) {
                        ed += 0.5 * p->L1 * Ds[k][d][i][j] * Ds[k][d][i][j] / cnt[k];
                        gDs[k][d][i][j] += p->L1 * Ds[k][d][i][j] / cnt[k];
                    }
                if (j == k) {
                    /* L2: D_j Q_ij D_j Q_ij ; L3: D_j Q_ij D_j Q_ij (same expression when j==k) */
                    for (int d = 0; d < 2; ++d)
                        if (ok[j][d]) {
                            ed += 0.5 * (p->L2 + p->L3) * Ds[j][d][i][j] * Ds[j][d][i][j] / cnt[j];
                            gDs[j][d][i][j] += (p->L2 + p->L3) * Ds[j][d][i][j] / cnt[j];
                        }
                } else {
                    ed += 0.5 * p->L2 * Dbar[j][i][j] * Dbar[k][i][k];
                    gDbar[j][i][j] += 0.5 * p->L2 * Dbar[k][i][k];
                    gDbar[k][i][k] += 0.5 * p->L2 * Dbar[j][i][j];
                    ed += 0.5 * p->L3 * Dbar[j][i][k] * Dbar[k][i][j];
                    gDbar[j][i][k] += 0.5 * p->L3 * Dbar[k][i][j];
                    gDbar[k][i][j] += 0.5 * p->L3 * Dbar[j][i][k];
                }
            }

    /* chiral term: linear in the differences, so its mean over the sign combinations is the same expression
     * on the mean differences Dbar */
    double gQ4[3][3];
    memset(gQ4, 0, sizeof(gQ4));
    if (p->L4 != 0.0)
        for (int l = 0; l < 3; ++l)
            for (int i = 0; i < 3; ++i)
                for (int k = 0; k < 3; ++k) {
                    const double e = eps3(l, i, k);
                    if (e == 0.0) continue;
                    for (int j = 0; j < 3; ++j) {
                        ed += 0.5 * p->L4 * e * Q[l][j] * Dbar[k][i][j];
                        gDbar[k][i][j] += 0.5 * p->L4 * e * Q[l][j];
                        gQ4[l][j] += 0.5 * p->L4 * e * Dbar[k][i][j];
                    }
                }

    /* cubic term L6/2 Q_lk D_l Q_ij D_k Q_ij: quadratic in the differences like the L1..L3 terms, so same-axis
     * products (l == k) average to the mean of squares and different-axis products to products of Dbar */
    if (p->L6 != 0.0)
        for (int l = 0; l < 3; ++l)
            for (int k = 0; k < 3; ++k)
                for (int i = 0; i < 3; ++i)
                    for (int j = 0; j < 3; ++j) {
                        if (l == k) {
                            for (int d = 0; d < 2; ++d)
                                if (ok[k][d]) {
                                    ed += 0.5 * p->L6 * Q[k][k] * Ds[k][d][i][j] * Ds[k][d][i][j] / cnt[k];
                                    gDs[k][d][i][j] += p->L6 * Q[k][k] * Ds[k][d][i][j] / cnt[k];
                                    gQ4[k][k] += 0.5 * p->L6 * Ds[k][d][i][j] * Ds[k][d][i][j] / cnt[k];
                                }
                        } else {
                            ed += 0.5 * p->L6 * Q[l][k] * Dbar[l][i][j] * Dbar[k][i][j];
                            gDbar[l][i][j] += 0.5 * p->L6 * Q[l][k] * Dbar[k][i][j];
                            gDbar[k][i][j] += 0.5 * p->L6 * Q[l][k] * Dbar[l][i][j];
                            gQ4[l][k] += 0.5 * p->L6 * Dbar[l][i][j] * Dbar[k][i][j];
                        }
                    }

    double eb = bulk_energy(p, Q) + field_energy(p, Q);      /* the "bulk" slot carries Eq. 13 too */
    double Ga[3][3];
    double ea = anchoring(p, N, s, is_boundary_site(p, x, y, z), Q, g ? Ga : NULL);

    if (g) {
        double G9[7][3][3];
        memset(G9, 0, sizeof(G9));
        bulk_grad(p, Q, G9[0]);
        field_grad_add(p, G9[0]);
        for (int i = 0; i < 3; ++i)
            for (int j = 0; j < 3; ++j) G9[0][i][j] += gQ4[i][j];
        for (int i = 0; i < 3; ++i)
            for (int j = 0; j < 3; ++j) G9[0][i][j] += Ga[i][j];
        for (int k = 0; k < 3; ++k)
            for (int d = 0; d < 2; ++d) {
                if (!ok[k][d]) continue;
                const int slot = 1 + 2 * k + d;
                for (int i = 0; i < 3; ++i)
                    for (int j = 0; j < 3; ++j) {
                        const double w = gDs[k][d][i][j] + gDbar[k][i][j] / cnt[k];
                        if (d == 0) { G9[slot][i][j] += w; G9[0][i][j] -= w; }
                        else        { G9[0][i][j] += w; G9[slot][i][j] -= w; }
                    }
            }
        for (int t = 0; t < 7; ++t) G_to_5(G9[t], g[t]);
    }
    if (terms) { terms[0] += eb; terms[1] += ed; terms[2] += ea; }
    return eb + ed + ea;
}

static double site_any(int variant, const lqo_problem *p, const double *q, int x, int y, int z,
                       double terms[3], double g[7][5])
{
    return variant == 0 ? site_literal(p, q, x, y, z, terms, g)
                        : site_factorised(p, q, x, y, z, terms, g);
}

/* single-site energy, exported for tests */
double lqo_site_energy(const lqo_problem *p, const double *q, int x, int y, int z, int variant, double terms[3])
{
    double t[3] = { 0, 0, 0 };
    double e = site_any(variant, p, q, x, y, z, t, NULL);
    if (terms) { terms[0] = t[0]; terms[1] = t[1]; terms[2] = t[2]; }
    return e;
}

/* ---------------------------------------------------------------- totals
 * F = sum over sites of f(x_i).  terms = (bulk, distortion,
 * anchoring) may be NULL.  long double accumulation so the result does not
 * depend on summation order at the 1e-9 level asked of the CUDA path.         */
double lqo_energy(const lqo_problem *p, const double *q, int variant, double terms[3])
{
    long double tb = 0.0L, td = 0.0L, ta = 0.0L;
    if (variant == 0) {
        for (int z = 0; z < p->Lz; ++z)
            for (int y = 0; y < p->Ly; ++y)
                for (int x = 0; x < p->Lx; ++x) {
                    double t[3] = { 0, 0, 0 };
                    site_literal(p, q, x, y, z, t, NULL);
                    tb += t[0]; td += t[1]; ta += t[2];
                }
    } else {
#pragma omp parallel for schedule(static) reduction(+ : tb, td, ta)
        for (int z = 0; z < p->Lz; ++z)
            for (int y = 0; y < p->Ly; ++y)
                for (int x = 0; x < p->Lx; ++x) {
                    double t[3] = { 0, 0, 0 };
                    site_factorised(p, q, x, y, z, t, NULL);
                    tb += t[0]; td += t[1]; ta += t[2];
                }
    }
    if (terms) { terms[0] = (double)tb; terms[1] = (double)td; terms[2] = (double)ta; }
    return (double)(tb + td + ta);
}

/* scatter the gradient of one site's energy into F (F = -dE/dq) */
static void scatter_site(int variant, const lqo_problem *p, const double *q, double *F, int x, int y, int z)
{
    const long N = (long)p->Lx * p->Ly * p->Lz;
    double g[7][5];
    if (!is_sim(p, site_of(p, x, y, z))) return;
    site_any(variant, p, q, x, y, z, NULL, g);
    long tgt[7];
    tgt[0] = site_of(p, x, y, z);
    for (int k = 0; k < 3; ++k) {
        tgt[1 + 2 * k] = nbr_of(p, x, y, z, k, +1);
        tgt[2 + 2 * k] = nbr_of(p, x, y, z, k, -1);
    }
    for (int t = 0; t < 7; ++t)
        for (int c = 0; c < 5; ++c) F[c * N + tgt[t]] -= g[t][c];
}

/* force field [5][N]; zero at object sites (they hold no variables) */
void lqo_forces(const lqo_problem *p, const double *q, double *F, int variant)
{
    const long N = (long)p->Lx * p->Ly * p->Lz;
    memset(F, 0, 5 * N * sizeof(double));
    if (variant == 0) {
        for (int z = 0; z < p->Lz; ++z)
            for (int y = 0; y < p->Ly; ++y)
                for (int x = 0; x < p->Lx; ++x) scatter_site(0, p, q, F, x, y, z);
        return;
    }
    /* a site in plane z writes planes z-1, z, z+1, so planes 3 apart never
     * collide: colour c handles z = c, c+3, ... below 3*floor(Lz/3) in
     * parallel (one thread per plane); the <= 2 left-over planes go serially. */
    const int zfull = 3 * (p->Lz / 3);
    for (int c = 0; c < 3; ++c) {
#pragma omp parallel for schedule(dynamic, 1)
        for (int z = c; z < zfull; z += 3)
            for (int y = 0; y < p->Ly; ++y)
                for (int x = 0; x < p->Lx; ++x) scatter_site(1, p, q, F, x, y, z);
    }
    for (int z = zfull; z < p->Lz; ++z)
        for (int y = 0; y < p->Ly; ++y)
            for (int x = 0; x < p->Lx; ++x) scatter_site(1, p, q, F, x, y, z);
}

/* force on ONE site: only the site's own energy and its 6 neighbours' energies
 * contain q(site) (each f(y) touches y and y +- k).  For sampled parity at
 * sizes where the full field is too slow.                                     */
void lqo_force_at(const lqo_problem *p, const double *q, int x, int y, int z, int variant, double F5[5])
{
    for (int c = 0; c < 5; ++c) F5[c] = 0.0;
    if (!is_sim(p, site_of(p, x, y, z))) return;
    double g[7][5];
    site_any(variant, p, q, x, y, z, NULL, g);
    for (int c = 0; c < 5; ++c) F5[c] -= g[0][c];
    for (int k = 0; k < 3; ++k)
        for (int sg = +1; sg >= -1; sg -= 2) {
            int xn = x, yn = y, zn = z;
            if (k == 0) xn = wrapi(x + sg, p->Lx);
            else if (k == 1) yn = wrapi(y + sg, p->Ly);
            else zn = wrapi(z + sg, p->Lz);
            if (!is_sim(p, site_of(p, xn, yn, zn))) continue;
            site_any(variant, p, q, xn, yn, zn, NULL, g);
            /* seen from the neighbour at +sg along k, our site is its -sg neighbour */
            const int slot = 1 + 2 * k + (sg > 0 ? 1 : 0);
            for (int c = 0; c < 5; ++c) F5[c] -= g[slot][c];
        }
}

/* ------------------------------------------------------------------- FIRE
 * Algorithm 1 with the readings DESIGN.md R3 (alpha is
 * multiplied by falpha < 1), R4 (velocity Verlet as kick-drift-kick), R12
 * (stop on max |F_a| < tol), R13 (state restarts per call, strict
 * Npos > Nmin, no dt floor, mixing skipped if |F|^2 == 0).  Unit mass.
 * q [5][N] in/out; v [5][N] out (may be NULL).  trace, if not NULL, receives
 * 8 doubles per step: dt, alpha, Npos, P, FF, vv, Fmax (all after the step's
 * schedule update except P,FF,vv,Fmax which are the step's reductions) and the
 * energy of the step's q if trace_energy != 0 (else 0).                       */
static void reduce4(const lqo_problem *p, const double *F, const double *v, long N,
                    double *P, double *FF, double *vv, double *Fmax)
{
    long double aP = 0.0L, aF = 0.0L, aV = 0.0L;
    double m = 0.0;
    for (int c = 0; c < 5; ++c) {
        long double bP = 0.0L, bF = 0.0L, bV = 0.0L;
        double bm = 0.0;
#pragma omp parallel for schedule(static) reduction(+ : bP, bF, bV) reduction(max : bm)
        for (long s = 0; s < N; ++s) {
            if (!is_sim(p, s)) continue;
            const double f = F[c * N + s], w = v[c * N + s];
            bP += (long double)f * w;
            bF += (long double)f * f;
            bV += (long double)w * w;
            const double af = fabs(f);
            if (af > bm) bm = af;
        }
        aP += bP; aF += bF; aV += bV;
        if (bm > m) m = bm;
    }
    *P = (double)aP; *FF = (double)aF; *vv = (double)aV; *Fmax = m;
}

int lqo_fire(const lqo_problem *p, double *q, double *v_out, long max_steps, double force_tol,
             const lqo_fire_params *fp, lqo_fire_report *rep, int variant,
             double *trace, int trace_energy)
{
    const long N = (long)p->Lx * p->Ly * p->Lz;
    long nsim = 0;
    for (long s = 0; s < N; ++s) nsim += is_sim(p, s);
    double *v = (double *)calloc(5 * N, sizeof(double));
    double *F = (double *)malloc(5 * N * sizeof(double));
    if (!v || !F) { free(v); free(F); return -4; }

    double dt = fp->dt0, alpha = fp->alpha0;
    int npos = 0;
    double P = 0.0, FF = 0.0, vv = 0.0, Fmax = 0.0;
    long step = 0;
    int converged = 0;

    lqo_forces(p, q, F, variant);
    reduce4(p, F, v, N, &P, &FF, &vv, &Fmax);
    if (Fmax < force_tol) converged = 1;

    /* integrator 1 (R30): FIRE on the plain semi-implicit Euler step,
     *     v += dt F(q);  P, |F|^2, |v|^2;  mix;  schedule;  q += dt v  (the step's dt, the mixed / reset v),
     * then the new force and the stop test; one force evaluation per step. */
    while (fp->integrator == 1 && !converged && step < max_steps) {
        ++step;
#pragma omp parallel for schedule(static)
        for (long i = 0; i < 5 * N; ++i) {
            if (!is_sim(p, i % N)) continue;
            v[i] += dt * F[i];
        }
        double Fm0;
        reduce4(p, F, v, N, &P, &FF, &vv, &Fm0);
        double dt_next = dt;
        if (FF > 0.0) {
            const double sc = alpha * sqrt(vv / FF);
#pragma omp parallel for schedule(static)
            for (long i = 0; i < 5 * N; ++i) {
                if (!is_sim(p, i % N)) continue;
                v[i] = (1.0 - alpha) * v[i] + sc * F[i];
            }
        }
        if (P > 0.0) {
            npos += 1;
            if (npos > fp->Nmin) {
                dt_next = fmin(dt * fp->finc, fp->dtmax);
                alpha *= fp->falpha;
            }
        } else {
            npos = 0;
            dt_next = dt * fp->fdec;
            alpha = fp->alpha0;
            memset(v, 0, 5 * N * sizeof(double));
        }
#pragma omp parallel for schedule(static)
        for (long i = 0; i < 5 * N; ++i) {
            if (!is_sim(p, i % N)) continue;
            q[i] += dt * v[i];
        }
        dt = dt_next;
        lqo_forces(p, q, F, variant);
        {
            double P1, FF1, vv1;
            reduce4(p, F, v, N, &P1, &FF1, &vv1, &Fmax);
            FF = FF1;                    /* reported Frms: of the force at the final q */
        }
        if (Fmax < force_tol) converged = 1;
        if (trace) {
            double *t = trace + 8 * (step - 1);
            t[0] = dt; t[1] = alpha; t[2] = (double)npos; t[3] = P; t[4] = FF; t[5] = vv; t[6] = Fmax;
            t[7] = trace_energy ? lqo_energy(p, q, variant, NULL) : 0.0;
        }
    }

    while (fp->integrator == 0 && !converged && step < max_steps) {
        ++step;
        /* velocity Verlet: half kick, drift, new force, half kick */
#pragma omp parallel for schedule(static)
        for (long i = 0; i < 5 * N; ++i) {
            if (!is_sim(p, i % N)) continue;
            v[i] += 0.5 * dt * F[i];
            q[i] += dt * v[i];
        }
        lqo_forces(p, q, F, variant);
#pragma omp parallel for schedule(static)
        for (long i = 0; i < 5 * N; ++i) {
            if (!is_sim(p, i % N)) continue;
            v[i] += 0.5 * dt * F[i];
        }
        /* power P = F.v and the norms used to rescale the velocity */
        reduce4(p, F, v, N, &P, &FF, &vv, &Fmax);
        if (Fmax < force_tol) converged = 1;
        if (!converged) {
            /* rescale velocity by alpha: v <- (1-alpha) v + alpha |v| F/|F| */
            if (FF > 0.0) {
                const double sc = alpha * sqrt(vv / FF);
#pragma omp parallel for schedule(static)
                for (long i = 0; i < 5 * N; ++i) {
                    if (!is_sim(p, i % N)) continue;
                    v[i] = (1.0 - alpha) * v[i] + sc * F[i];
                }
            }
            if (P > 0.0) {
                npos += 1;
                if (npos > fp->Nmin) {
                    dt = fmin(dt * fp->finc, fp->dtmax);
                    alpha *= fp->falpha;
                }
            } else {
                npos = 0;
                dt *= fp->fdec;
                alpha = fp->alpha0;
                memset(v, 0, 5 * N * sizeof(double));
            }
        }
        if (trace) {
            double *t = trace + 8 * (step - 1);
            t[0] = dt; t[1] = alpha; t[2] = (double)npos; t[3] = P; t[4] = FF; t[5] = vv; t[6] = Fmax;
            t[7] = trace_energy ? lqo_energy(p, q, variant, NULL) : 0.0;
        }
    }
    if (rep) {
        rep->steps = step; rep->converged = converged;
        rep->Fmax = Fmax; rep->Frms = nsim ? sqrt(FF / (double)nsim) : 0.0;
        rep->P = P; rep->dt = dt; rep->alpha = alpha;
        rep->energy = lqo_energy(p, q, variant, NULL);
    }
    if (v_out) memcpy(v_out, v, 5 * N * sizeof(double));
    free(v); free(F);
    return 0;
}

/* ------------------------------------------- gradient descent and Nesterov
 * the paper's comparator minimiser (gradient descent, PAPER.md:189,
 * 205-211, "steepest descent relaxation ... overdamped molecular dynamics at zero
 * temperature") and its second GUI minimiser (Nesterov's accelerated gradient,
 * PAPER.md:189, 289, 445).  The paper gives neither formula nor parameters; the
 * readings (R23, R24) are the textbook fixed-step forms:
 *   method 0 (GD):        y_k = q_k
 *   method 1 (Nesterov):  y_k = q_k + mu (q_k - q_{k-1}),   q_{-1} = q_0   [80]
 *   q_{k+1} = y_k + eta F(y_k),   F = -dF/dq
 * on simulated sites only; object sites never move.  Stop (R12) when
 * max |F_a(y_k)| < force_tol; the step that measured it is still applied (its
 * update is a by-product of the same pass), so steps = number of updates applied.
 * trace, if not NULL, gets 3 doubles per step: |F|^2, max|F_a| of F(y_k), and the
 * energy of q_{k+1} if trace_energy (else 0).                                    */
int lqo_descent(const lqo_problem *p, double *q, int method, long max_steps, double force_tol,
                double eta, double mu, lqo_fire_report *rep, int variant, double *trace, int trace_energy)
{
    const long N = (long)p->Lx * p->Ly * p->Lz;
    long nsim = 0;
    for (long s = 0; s < N; ++s) nsim += is_sim(p, s);
    double *F = (double *)malloc(5 * N * sizeof(double));
    double *y = (double *)malloc(5 * N * sizeof(double));
    double *qprev = (double *)malloc(5 * N * sizeof(double));
    double *zero = (double *)calloc(5 * N, sizeof(double));
    if (!F || !y || !qprev || !zero) { free(F); free(y); free(qprev); free(zero); return -4; }
    memcpy(qprev, q, 5 * N * sizeof(double));
    double P = 0.0, FF = 0.0, vv = 0.0, Fmax = 0.0;
    long step = 0;
    int converged = 0;
    while (!converged && step < max_steps) {
        ++step;
        for (long i = 0; i < 5 * N; ++i) {
            y[i] = q[i];
            if (method == 1 && is_sim(p, i % N)) y[i] = q[i] + mu * (q[i] - qprev[i]);
        }
        lqo_forces(p, y, F, variant);
        reduce4(p, F, zero, N, &P, &FF, &vv, &Fmax);
        if (Fmax < force_tol) converged = 1;
        memcpy(qprev, q, 5 * N * sizeof(double));
        for (long i = 0; i < 5 * N; ++i) {
            if (!is_sim(p, i % N)) continue;
            q[i] = y[i] + eta * F[i];
        }
        if (trace) {
            double *t = trace + 3 * (step - 1);
            t[0] = FF; t[1] = Fmax; t[2] = trace_energy ? lqo_energy(p, q, variant, NULL) : 0.0;
        }
    }
    if (rep) {
        rep->steps = step; rep->converged = converged;
        rep->Fmax = Fmax; rep->Frms = nsim ? sqrt(FF / (double)nsim) : 0.0;
        rep->P = 0.0; rep->dt = eta; rep->alpha = mu;
        rep->energy = lqo_energy(p, q, variant, NULL);
    }
    free(F); free(y); free(qprev); free(zero);
    return 0;
}

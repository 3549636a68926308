// lq_site.cuh -- per-site Landau-de Gennes arithmetic in GATHER form (device functions).
//
// The force on the five stored variables of site x is assembled from the 3x3 gradient
// G_ab = dF/dQ_ab (entries treated as independent), F = -(Gxx-Gzz, Gxy+Gyx, Gxz+Gzx,
// Gyy-Gzz, Gyz+Gzy).  Derivation of every piece: DESIGN.md section 6.
//   bulk      Eq. 5:   G = (A + C tr Q^2) Q + B Q^2
//   elastic   Eq. 10 averaged over the allowed forward/backward differences
//             (PAPER.md:177-183).  With a^s_k(y) = "y + s k is simulated",
//             w_k(y) = 1/(a+_k + a-_k) (0 if none), Dbar_k = w_k * sum_s a^s_k D^s_k:
//       same-axis:  G_ab(x) -= sum_k (L1 + (L2+L3) d_bk) sum_s a^s_k(x) [w_k(x) + w_k(x+s k)] (Q_ab(x+s k) - Q_ab(x))
//       mixed:      H^(c)_ab(y) = L2 d_bc sum_{m!=c} Dbar_m Q_am(y) + L3 (1-d_bc) Dbar_b Q_ac(y)
//                   G_ab(x) += sum_c { w_c(x)(a-_c(x) - a+_c(x)) H^(c)_ab(x)
//                                      + a-_c(x) w_c(x-c) H^(c)_ab(x-c) - a+_c(x) w_c(x+c) H^(c)_ab(x+c) }
//   anchoring Eq. 14: G += 2W (Q - Q0), Q0 = 3/2 S0 (n n - I/3)
//             Eq. 15: G += 2W M, M = Qt - P Qt P, Qt = Q + S0/2 I, P = I - nu nu
// An accessor type supplies Q (6 numbers xx,xy,xz,yy,yz,zz) and the flag byte at small
// offsets from the site, so the same code serves global-memory and shared-memory tiles.
#pragma once
#include "lq_internal.cuh"

namespace lqs {

__device__ __forceinline__ int m6(int a, int b) {
    // index of tensor entry (a,b) in (xx,xy,xz,yy,yz,zz)
    return a == b ? (a == 0 ? 0 : (a == 1 ? 3 : 5)) : (a + b == 1 ? 1 : (a + b == 2 ? 2 : 4));
}
__device__ __forceinline__ int a_plus(unsigned fl, int k) { return (fl >> (2 + 2 * k)) & 1u; }
__device__ __forceinline__ int a_minus(unsigned fl, int k) { return (fl >> (3 + 2 * k)) & 1u; }
__device__ __forceinline__ double w_axis(unsigned fl, int k) {
    const int n = a_plus(fl, k) + a_minus(fl, k);
    return n == 2 ? 0.5 : (n == 1 ? 1.0 : 0.0);
}

// accessor over padded global arrays, centred on padded index p
struct GlobalAcc {
    const double *q;
    const uint8_t *flags;  // may be null: every site bulk with all neighbours simulated
    long long NP, sy, sz, p;
    __device__ __forceinline__ void Q(int dx, int dy, int dz, double o[6]) const {
        const long long i = p + dx + dy * sy + dz * sz;
        o[0] = q[i]; o[1] = q[NP + i]; o[2] = q[2 * NP + i]; o[3] = q[3 * NP + i]; o[4] = q[4 * NP + i];
        o[5] = -o[0] - o[3];
    }
    __device__ __forceinline__ unsigned flag(int dx, int dy, int dz) const {
        return flags ? (unsigned)flags[p + dx + dy * sy + dz * sz] : 0xFCu;
    }
};

__device__ __forceinline__ void off3(int k, int s, int &dx, int &dy, int &dz) {
    dx = k == 0 ? s : 0; dy = k == 1 ? s : 0; dz = k == 2 ? s : 0;
}

// Dbar_m Q at the site at offset (ox,oy,oz), whose flag byte is fl and tensor is Qy
template <class Acc>
__device__ __forceinline__ void dbar(const Acc &acc, int ox, int oy, int oz, unsigned fl, const double Qy[6],
                                     int m, double out[6]) {
    const int ap = a_plus(fl, m), am = a_minus(fl, m);
    const double w = w_axis(fl, m);
    int dx, dy, dz;
    double t[6];
#pragma unroll
    for (int i = 0; i < 6; ++i) out[i] = 0.0;
    if (ap) {
        off3(m, +1, dx, dy, dz);
        acc.Q(ox + dx, oy + dy, oz + dz, t);
#pragma unroll
        for (int i = 0; i < 6; ++i) out[i] += t[i] - Qy[i];
    }
    if (am) {
        off3(m, -1, dx, dy, dz);
        acc.Q(ox + dx, oy + dy, oz + dz, t);
#pragma unroll
        for (int i = 0; i < 6; ++i) out[i] += Qy[i] - t[i];
    }
#pragma unroll
    for (int i = 0; i < 6; ++i) out[i] *= w;
}

__device__ __forceinline__ void bulk_G(const LqPhys &ph, const double Q[6], double G[3][3]) {
    const double a = Q[0], b = Q[1], c = Q[2], d = Q[3], e = Q[4], f = Q[5];
    const double q2xx = a * a + b * b + c * c, q2xy = a * b + b * d + c * e, q2xz = a * c + b * e + c * f;
    const double q2yy = b * b + d * d + e * e, q2yz = b * c + d * e + e * f, q2zz = c * c + e * e + f * f;
    const double k = ph.A + ph.C * (q2xx + q2yy + q2zz);
    // - T_ab: the external-field term of Eq. 13 (constant; folds into the FMAs, exact no-op when T = 0)
    G[0][0] = k * a + (ph.B * q2xx - ph.T[0]); G[0][1] = G[1][0] = k * b + (ph.B * q2xy - ph.T[1]);
    G[0][2] = G[2][0] = k * c + (ph.B * q2xz - ph.T[2]); G[1][1] = k * d + (ph.B * q2yy - ph.T[3]);
    G[1][2] = G[2][1] = k * e + (ph.B * q2yz - ph.T[4]); G[2][2] = k * f + (ph.B * q2zz - ph.T[5]);
}

__device__ __forceinline__ double bulk_E(const LqPhys &ph, const double Q[6]) {
    const double a = Q[0], b = Q[1], c = Q[2], d = Q[3], e = Q[4], f = Q[5];
    const double q2xx = a * a + b * b + c * c, q2xy = a * b + b * d + c * e, q2xz = a * c + b * e + c * f;
    const double q2yy = b * b + d * d + e * e, q2yz = b * c + d * e + e * f, q2zz = c * c + e * e + f * f;
    const double tr2 = q2xx + q2yy + q2zz;
    const double tr3 = q2xx * a + q2yy * d + q2zz * f + 2.0 * (q2xy * b + q2xz * c + q2yz * e);
    const double fext = -(ph.T[0] * a + ph.T[3] * d + ph.T[5] * f + 2.0 * (ph.T[1] * b + ph.T[2] * c + ph.T[4] * e));   // Eq. 13
    return 0.5 * ph.A * tr2 + ph.B * (1.0 / 3.0) * tr3 + 0.25 * ph.C * tr2 * tr2 + fext;
}

// anchoring: adds to G (if G != nullptr) and returns the energy
__device__ __forceinline__ double anchoring(const LqPhys &ph, int kind, double W, const double n[3],
                                            const double Q[6], double (*G)[3]) {
    double e = 0.0;
    if (kind == 1) {
        const double q0 = 1.5 * ph.S0;
#pragma unroll
        for (int a = 0; a < 3; ++a)
#pragma unroll
            for (int b = 0; b < 3; ++b) {
                const double d = Q[m6(a, b)] - q0 * (n[a] * n[b] - (a == b ? 1.0 / 3.0 : 0.0));
                e += W * d * d;
                if (G) G[a][b] += 2.0 * W * d;
            }
    } else if (kind == 2) {
        // M = Qt - P Qt P with P = I - nu nu:  M = nu u^T + u nu^T - s nu nu^T, u = Qt nu, s = nu.Qt.nu
        double u[3];
        const double h = 0.5 * ph.S0;
#pragma unroll
        for (int a = 0; a < 3; ++a)
            u[a] = Q[m6(a, 0)] * n[0] + Q[m6(a, 1)] * n[1] + Q[m6(a, 2)] * n[2] + h * n[a];
        const double s = u[0] * n[0] + u[1] * n[1] + u[2] * n[2];
#pragma unroll
        for (int a = 0; a < 3; ++a)
#pragma unroll
            for (int b = 0; b < 3; ++b) {
                const double M = n[a] * u[b] + u[a] * n[b] - s * n[a] * n[b];
                e += W * M * M;
                if (G) G[a][b] += 2.0 * W * M;
            }
    }
    return e;
}

// Frobenius product of two symmetric tensors stored as (xx, xy, xz, yy, yz, zz)
__device__ __forceinline__ double frodot(const double a[6], const double b[6]) {
    return a[0] * b[0] + a[3] * b[3] + a[5] * b[5] + 2.0 * (a[1] * b[1] + a[2] * b[2] + a[4] * b[4]);
}

__device__ __forceinline__ void G_to_F(const double G[3][3], double F[5]) {
    F[0] = -(G[0][0] - G[2][2]);
    F[1] = -(G[0][1] + G[1][0]);
    F[2] = -(G[0][2] + G[2][0]);
    F[3] = -(G[1][1] - G[2][2]);
    F[4] = -(G[1][2] + G[2][1]);
}

// Force on a simulated site in the general (masked, L1/L2/L3, anchored) case.
// fl = the site's flag byte; akind/W/n = its anchoring record (akind 0 if none).
template <bool THREE, class Acc>
__device__ __forceinline__ void site_force(const LqPhys &ph, const Acc &acc, unsigned fl, int akind, double W,
                                           const double n[3], double F[5]) {
    double Qx[6], G[3][3];
    acc.Q(0, 0, 0, Qx);
    bulk_G(ph, Qx, G);
    if ((fl & 3u) == 1u && akind != 0) anchoring(ph, akind, W, n, Qx, G);
    const double L23 = ph.L2 + ph.L3;
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        const double wx = w_axis(fl, k);
#pragma unroll
        for (int s = +1; s >= -1; s -= 2) {
            const int allowed = s > 0 ? a_plus(fl, k) : a_minus(fl, k);
            if (!allowed) continue;
            int dx, dy, dz;
            off3(k, s, dx, dy, dz);
            const unsigned fn = acc.flag(dx, dy, dz);
            const double wn = w_axis(fn, k);
            const double coef = wx + wn;
            double Qn[6];
            acc.Q(dx, dy, dz, Qn);
            // cubic term, same-axis part: the bond weight of L1 with Q_kk w_k of the bond's two ends (Eq. 10, L6)
            const double c6 = THREE ? ph.L6 * (wx * Qx[m6(k, k)] + wn * Qn[m6(k, k)]) : 0.0;
#pragma unroll
            for (int a = 0; a < 3; ++a)
#pragma unroll
                for (int b = 0; b < 3; ++b) {
                    const double cab = ph.L1 + ((THREE && b == k) ? L23 : 0.0);
                    G[a][b] -= (cab * coef + c6) * (Qn[m6(a, b)] - Qx[m6(a, b)]);
                }
            if (THREE && ph.L6 != 0.0) {
                // ... and its undifferentiated factor Q_kk(x): d/dQ_kk(x) = L6/2 w_k(x) |D^s_k Q(x)|^2
                double D[6];
#pragma unroll
                for (int i = 0; i < 6; ++i) D[i] = Qn[i] - Qx[i];
                G[k][k] += 0.5 * ph.L6 * wx * frodot(D, D);
            }
        }
    }
    if (THREE) {
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            const int m1 = (c + 1) % 3, m2 = (c + 2) % 3;
#pragma unroll
            for (int t = 0; t < 3; ++t) {
                // t = 0: y = x;  t = 1: y = x - c;  t = 2: y = x + c
                int ox = 0, oy = 0, oz = 0;
                double coef;
                unsigned fy;
                if (t == 0) {
                    coef = w_axis(fl, c) * (double)(a_minus(fl, c) - a_plus(fl, c));
                    fy = fl;
                } else {
                    const int s = t == 1 ? -1 : +1;
                    const int allowed = s > 0 ? a_plus(fl, c) : a_minus(fl, c);
                    if (!allowed) continue;
                    off3(c, s, ox, oy, oz);
                    fy = acc.flag(ox, oy, oz);
                    coef = (s > 0 ? -1.0 : 1.0) * w_axis(fy, c);
                }
                if (coef == 0.0) continue;
                double Qy[6], D1[6], D2[6];
                acc.Q(ox, oy, oz, Qy);
                dbar(acc, ox, oy, oz, fy, Qy, m1, D1);
                dbar(acc, ox, oy, oz, fy, Qy, m2, D2);
#pragma unroll
                for (int a = 0; a < 3; ++a) {
                    G[a][c] += coef * ph.L2 * (D1[m6(a, m1)] + D2[m6(a, m2)]);
                    G[a][m1] += coef * ph.L3 * D1[m6(a, c)];
                    G[a][m2] += coef * ph.L3 * D2[m6(a, c)];
                }
                // chiral term: H^(c)_ab(y) = d f4(y) / d(Dbar_c Q_ab) = L4/2 eps_lac Q_lb(y)
#pragma unroll
                for (int b = 0; b < 3; ++b) {
                    G[m2][b] += coef * 0.5 * ph.L4 * Qy[m6(m1, b)];
                    G[m1][b] -= coef * 0.5 * ph.L4 * Qy[m6(m2, b)];
                }
                // cubic term, mixed part: H^(c)_ab(y) = L6 sum_{l != c} Q_lc(y) Dbar_l Q_ab(y)
                if (ph.L6 != 0.0) {
                    const double h1 = coef * ph.L6 * Qy[m6(m1, c)], h2 = coef * ph.L6 * Qy[m6(m2, c)];
#pragma unroll
                    for (int a = 0; a < 3; ++a)
#pragma unroll
                        for (int b = 0; b < 3; ++b) G[a][b] += h1 * D1[m6(a, b)] + h2 * D2[m6(a, b)];
                }
            }
        }
        if (ph.L4 != 0.0 || ph.L6 != 0.0) {
            // ... and its undifferentiated factor: d f4(x) / dQ_ab(x) = L4/2 eps_aik Dbar_k Q_ib(x)
            double Dk[3][6];
#pragma unroll
            for (int k = 0; k < 3; ++k) dbar(acc, 0, 0, 0, fl, Qx, k, Dk[k]);
#pragma unroll
            for (int a = 0; a < 3; ++a) {
                const int a1 = (a + 1) % 3, a2 = (a + 2) % 3;
#pragma unroll
                for (int b = 0; b < 3; ++b) G[a][b] += 0.5 * ph.L4 * (Dk[a2][m6(a1, b)] - Dk[a1][m6(a2, b)]);
                // cubic term, undifferentiated off-diagonal factor: d/dQ_ab(x) = L6/2 Dbar_a Q : Dbar_b Q  (a != b)
                G[a][a1] += 0.5 * ph.L6 * frodot(Dk[a], Dk[a1]);
                G[a][a2] += 0.5 * ph.L6 * frodot(Dk[a], Dk[a2]);
            }
        }
    }
    G_to_F(G, F);
}

// Energy of one simulated site: terms = (bulk, distortion, anchoring)
template <bool THREE, class Acc>
__device__ __forceinline__ void site_energy(const LqPhys &ph, const Acc &acc, unsigned fl, int akind, double W,
                                            const double n[3], double terms[3]) {
    double Qx[6];
    acc.Q(0, 0, 0, Qx);
    terms[0] = bulk_E(ph, Qx);
    terms[2] = ((fl & 3u) == 1u && akind != 0) ? anchoring(ph, akind, W, n, Qx, nullptr) : 0.0;
    const double L23 = ph.L2 + ph.L3;
    double ed = 0.0;
    double Db[3][6];
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        const double w = w_axis(fl, k);
#pragma unroll
        for (int i = 0; i < 6; ++i) Db[k][i] = 0.0;
#pragma unroll
        for (int s = +1; s >= -1; s -= 2) {
            const int allowed = s > 0 ? a_plus(fl, k) : a_minus(fl, k);
            if (!allowed) continue;
            int dx, dy, dz;
            off3(k, s, dx, dy, dz);
            double Qn[6], D[6];
            acc.Q(dx, dy, dz, Qn);
#pragma unroll
            for (int i = 0; i < 6; ++i) {
                D[i] = s > 0 ? Qn[i] - Qx[i] : Qx[i] - Qn[i];
                Db[k][i] += w * D[i];
            }
            const double fro = D[0] * D[0] + D[3] * D[3] + D[5] * D[5] + 2.0 * (D[1] * D[1] + D[2] * D[2] + D[4] * D[4]);
            ed += 0.5 * ph.L1 * w * fro;
            if (THREE) {
                const double col = D[m6(0, k)] * D[m6(0, k)] + D[m6(1, k)] * D[m6(1, k)] + D[m6(2, k)] * D[m6(2, k)];
                ed += 0.5 * L23 * w * col;
                ed += 0.5 * ph.L6 * Qx[m6(k, k)] * w * fro;          // cubic term, same-axis part
            }
        }
    }
    if (THREE) {
#pragma unroll
        for (int j = 0; j < 3; ++j)
#pragma unroll
            for (int k = j + 1; k < 3; ++k)
#pragma unroll
                for (int i = 0; i < 3; ++i) {
                    ed += ph.L2 * Db[j][m6(i, j)] * Db[k][m6(i, k)];
                    ed += ph.L3 * Db[j][m6(i, k)] * Db[k][m6(i, j)];
                }
        // cubic term, mixed part: L6/2 sum_{l != k} Q_lk Dbar_l Q : Dbar_k Q
#pragma unroll
        for (int j = 0; j < 3; ++j)
#pragma unroll
            for (int k = j + 1; k < 3; ++k) ed += ph.L6 * Qx[m6(j, k)] * frodot(Db[j], Db[k]);
        // chiral term L4/2 eps_lik Q_lj Dbar_k Q_ij: for axis k the pairs (l, i) = (k+1, k+2) [+1] and (k+2, k+1) [-1]
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            const int k1 = (k + 1) % 3, k2 = (k + 2) % 3;
#pragma unroll
            for (int j = 0; j < 3; ++j)
                ed += 0.5 * ph.L4 * (Qx[m6(k1, j)] * Db[k][m6(k2, j)] - Qx[m6(k2, j)] * Db[k][m6(k1, j)]);
        }
    }
    terms[1] = ed;
}

// one-constant, pure-bulk neighbourhood: F from the centre tensor and the 7-point Laplacian
// lap[c] = sum over the 6 neighbours of (q_c(nbr) - q_c(x))      (Eq. 11)
__device__ __forceinline__ void bulk_force_oneconst(const LqPhys &ph, const double q5[5], const double lap[5],
                                                    double F[5]) {
    double Q[6] = {q5[0], q5[1], q5[2], q5[3], q5[4], -q5[0] - q5[3]};
    double G[3][3];
    bulk_G(ph, Q, G);
    F[0] = -(G[0][0] - G[2][2]) + ph.L1 * (2.0 * lap[0] + lap[3]);
    F[1] = -2.0 * G[0][1] + 2.0 * ph.L1 * lap[1];
    F[2] = -2.0 * G[0][2] + 2.0 * ph.L1 * lap[2];
    F[3] = -(G[1][1] - G[2][2]) + ph.L1 * (2.0 * lap[3] + lap[0]);
    F[4] = -2.0 * G[1][2] + 2.0 * ph.L1 * lap[4];
}

// three-constant, pure-bulk neighbourhood (19-point).  get(c, dx, dy, dz) returns stored component c at an
// offset with |dx|+|dy|+|dz| <= 2 and at most two non-zero entries.  With T_ab the elastic part of -G_ab,
//   T_ab = L1 lap(Q_ab) + (L2+L3) [ d2_b(Q_ab) + sum_{m != b} X_bm(Q_am) ],
//   X_bm f = 1/4 [f(+b+m) - f(+b-m) - f(-b+m) + f(-b-m)]   (bulk specialisation)
// and Qzz = -Qxx - Qyy eliminated by linearity:
//   F0 = L1(2 lap xx + lap yy) + L23[d2x xx + d2z xx + d2z yy + Xxy xy - Xyz yz]
//   F3 = L1(2 lap yy + lap xx) + L23[d2y yy + d2z xx + d2z yy + Xxy xy - Xxz xz]
//   F1 = 2 L1 lap xy + L23[d2x xy + d2y xy + Xxy xx + Xxy yy + Xyz xz + Xxz yz]
//   F2 = 2 L1 lap xz + L23[d2x xz + d2z xz + Xyz xy + Xxy yz - Xxz yy]
//   F4 = 2 L1 lap yz + L23[d2y yz + d2z yz + Xxz xy + Xxy xz - Xyz xx]
// CHIRAL: also the L4 term on constant weights, G_ab += L4 eps_aik C_k Q_ib with centred differences C_k (the
// gather form of lqs::site_force at a site whose weights are all 1/2) -- a template flag so
// that the achiral instantiations keep their register budget.
// CUBIC: the L6 term on constant weights (all w = 1/2), from the same gather form:
//   bonds      G_ab -= L6/2 [Q_kk(x) + Q_kk(x + s k)] (Q_ab(x + s k) - Q_ab(x))            for the six neighbours
//   own factor G_kk += L6/4 sum_s |Q(x + s k) - Q(x)|^2 ;  G_ab += L6/2 C_a Q : C_b Q  (a != b)
//   mixed      G_ab += sum_c 1/2 [H_c(x - c) - H_c(x + c)]_ab ,  H_c(y) = L6 sum_{l != c} Q_lc(y) C_l Q(y)
// with C_l the centred difference; the edge neighbours x +- c +- l enter through C_l Q(x +- c).
template <bool CHIRAL = false, bool CUBIC = false, class Get>
__device__ __forceinline__ void bulk_force_threeconst(const LqPhys &ph, const Get &g, const double qc[5], double F[5]) {
    const double L1 = ph.L1, L23 = ph.L2 + ph.L3;
    auto d2 = [&](int c, int ax) -> double {
        return (g(c, ax == 0, ax == 1, ax == 2) + g(c, -(ax == 0), -(ax == 1), -(ax == 2))) - 2.0 * qc[c];
    };
    auto X = [&](int c, int b, int m) -> double {   // axes b < m
        const int bx = b == 0, by = b == 1, bz = b == 2, mx = m == 0, my = m == 1, mz = m == 2;
        return 0.25 * ((g(c, bx + mx, by + my, bz + mz) - g(c, bx - mx, by - my, bz - mz)) -
                       (g(c, -bx + mx, -by + my, -bz + mz) - g(c, -bx - mx, -by - my, -bz - mz)));
    };
    double Q[6] = {qc[0], qc[1], qc[2], qc[3], qc[4], -qc[0] - qc[3]};
    double G[3][3];
    bulk_G(ph, Q, G);
    F[0] = -(G[0][0] - G[2][2]); F[1] = -2.0 * G[0][1]; F[2] = -2.0 * G[0][2];
    F[3] = -(G[1][1] - G[2][2]); F[4] = -2.0 * G[1][2];
    {   // xx: lap, d2x, d2z, Xxy, Xyz
        const double dx = d2(0, 0), dy = d2(0, 1), dz = d2(0, 2), lap = dx + dy + dz;
        F[0] += 2.0 * L1 * lap + L23 * (dx + dz);
        F[3] += L1 * lap + L23 * dz;
        F[1] += L23 * X(0, 0, 1);
        F[4] -= L23 * X(0, 1, 2);
    }
    {   // yy: lap, d2y, d2z, Xxy, Xxz
        const double dx = d2(3, 0), dy = d2(3, 1), dz = d2(3, 2), lap = dx + dy + dz;
        F[3] += 2.0 * L1 * lap + L23 * (dy + dz);
        F[0] += L1 * lap + L23 * dz;
        F[1] += L23 * X(3, 0, 1);
        F[2] -= L23 * X(3, 0, 2);
    }
    {   // xy: lap, d2x, d2y, Xxy, Xxz, Xyz
        const double dx = d2(1, 0), dy = d2(1, 1), dz = d2(1, 2), lap = dx + dy + dz;
        F[1] += 2.0 * L1 * lap + L23 * (dx + dy);
        const double xxy = X(1, 0, 1);
        F[0] += L23 * xxy;
        F[3] += L23 * xxy;
        F[4] += L23 * X(1, 0, 2);
        F[2] += L23 * X(1, 1, 2);
    }
    {   // xz: lap, d2x, d2z, Xxy, Xxz, Xyz
        const double dx = d2(2, 0), dy = d2(2, 1), dz = d2(2, 2), lap = dx + dy + dz;
        F[2] += 2.0 * L1 * lap + L23 * (dx + dz);
        F[4] += L23 * X(2, 0, 1);
        F[3] -= L23 * X(2, 0, 2);
        F[1] += L23 * X(2, 1, 2);
    }
    {   // yz: lap, d2y, d2z, Xxy, Xxz, Xyz
        const double dx = d2(4, 0), dy = d2(4, 1), dz = d2(4, 2), lap = dx + dy + dz;
        F[4] += 2.0 * L1 * lap + L23 * (dy + dz);
        F[2] += L23 * X(4, 0, 1);
        F[1] += L23 * X(4, 0, 2);
        F[0] -= L23 * X(4, 1, 2);
    }
    if (CHIRAL) {
        double Cd[3][6];                 // C_k of (xx, xy, xz, yy, yz, zz)
#pragma unroll
        for (int k = 0; k < 3; ++k) {
#pragma unroll
            for (int c = 0; c < 5; ++c)
                Cd[k][c] = 0.5 * (g(c, k == 0, k == 1, k == 2) - g(c, -(k == 0), -(k == 1), -(k == 2)));
            Cd[k][5] = -Cd[k][0] - Cd[k][3];
        }
        double G4[3][3];
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            const int a1 = (a + 1) % 3, a2 = (a + 2) % 3;
#pragma unroll
            for (int b = 0; b < 3; ++b) G4[a][b] = ph.L4 * (Cd[a2][m6(a1, b)] - Cd[a1][m6(a2, b)]);
        }
        F[0] -= G4[0][0] - G4[2][2]; F[1] -= G4[0][1] + G4[1][0]; F[2] -= G4[0][2] + G4[2][0];
        F[3] -= G4[1][1] - G4[2][2]; F[4] -= G4[1][2] + G4[2][1];
    }
    if (CUBIC) {
        auto T6 = [&](int dx, int dy, int dz, double o[6]) {     // full tensor at an offset
#pragma unroll
            for (int c = 0; c < 5; ++c) o[c] = g(c, dx, dy, dz);
            o[5] = -o[0] - o[3];
        };
        const double Q0[6] = {qc[0], qc[1], qc[2], qc[3], qc[4], -qc[0] - qc[3]};
        double G6[3][3] = {{0.0, 0.0, 0.0}, {0.0, 0.0, 0.0}, {0.0, 0.0, 0.0}};
        double Cx[3][6];                                         // C_k Q at the site itself
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            const int ex = k == 0, ey = k == 1, ez = k == 2;
            const int m1 = (k + 1) % 3, m2 = (k + 2) % 3;
            double Qp[6], Qm[6];
            T6(ex, ey, ez, Qp);
            T6(-ex, -ey, -ez, Qm);
            double dp[6], dm[6];
#pragma unroll
            for (int i = 0; i < 6; ++i) { dp[i] = Qp[i] - Q0[i]; dm[i] = Qm[i] - Q0[i]; Cx[k][i] = 0.5 * (Qp[i] - Qm[i]); }
            const double wp = 0.5 * ph.L6 * (Q0[m6(k, k)] + Qp[m6(k, k)]), wm = 0.5 * ph.L6 * (Q0[m6(k, k)] + Qm[m6(k, k)]);
#pragma unroll
            for (int a = 0; a < 3; ++a)
#pragma unroll
                for (int b = 0; b < 3; ++b) G6[a][b] -= wp * dp[m6(a, b)] + wm * dm[m6(a, b)];
            G6[k][k] += 0.25 * ph.L6 * (frodot(dp, dp) + frodot(dm, dm));
            // mixed part: y = x + s k, l in {m1, m2}
#pragma unroll
            for (int s = -1; s <= 1; s += 2) {
                const double *Qy = s > 0 ? Qp : Qm;
                double H[6] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
#pragma unroll
                for (int t = 0; t < 2; ++t) {
                    const int l = t == 0 ? m1 : m2;
                    const int lx = l == 0, ly = l == 1, lz = l == 2;
                    double A[6], Bm[6];
                    T6(s * ex + lx, s * ey + ly, s * ez + lz, A);
                    T6(s * ex - lx, s * ey - ly, s * ez - lz, Bm);
                    const double wl = ph.L6 * Qy[m6(l, k)] * 0.5;
#pragma unroll
                    for (int i = 0; i < 6; ++i) H[i] += wl * (A[i] - Bm[i]);
                }
                // 1/2 [H(x - k) - H(x + k)]
#pragma unroll
                for (int a = 0; a < 3; ++a)
#pragma unroll
                    for (int b = 0; b < 3; ++b) G6[a][b] += (s > 0 ? -0.5 : 0.5) * H[m6(a, b)];
            }
        }
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            const int a1 = (a + 1) % 3, a2 = (a + 2) % 3;
            G6[a][a1] += 0.5 * ph.L6 * frodot(Cx[a], Cx[a1]);
            G6[a][a2] += 0.5 * ph.L6 * frodot(Cx[a], Cx[a2]);
        }
        F[0] -= G6[0][0] - G6[2][2]; F[1] -= G6[0][1] + G6[1][0]; F[2] -= G6[0][2] + G6[2][0];
        F[3] -= G6[1][1] - G6[2][2]; F[4] -= G6[1][2] + G6[2][1];
    }
}

}  // namespace lqs

/*
 * mlmd_ref.c -- FP64 CPU ORACLE for the domain-batched real-time Kohn-Sham step.
 *
 * TEST INFRASTRUCTURE ONLY.  This file is the slow, plain, obviously-correct statement of
 * what the hot path computes.  It shares no code, header, table or constant with the CUDA
 * library under paper_2509_00966_b200/csrc/ and is never linked into or called from it.
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
 * may load it.
 *
 * What it computes (citations: PAPER.md line / equation; BASELINE.json north_star; DESIGN.md
 * reading numbers D1..D26 which restate SURVEY.md section 8(c)):
 *
 *   H = 1/2 (-i grad + A)^2 + V_loc + V_NL                     PAPER.md Eq. (3); a.u. (D6)
 *     = -1/2 D2  - i A.D1  + 1/2 |A|^2  + V_loc(r)  +  dv * B diag(D) B^H       (D5, D10)
 *   D2, D1: independent 4th-order central differences, periodic in x,y,z       north_star; D3, D26
 *       c2 = [-1/12, 4/3, -5/2, 4/3, -1/12] / h^2 ,  c1 = [1/12, -2/3, 0, 2/3, -1/12] / h
 *   V_NL psi = sum_p beta_p D_p <beta_p|psi>,  <a|b> = dv * sum_r conj(a) b     north_star; D4, D10
 *   one step:  psi <- sum_{m=0..4} (-i dt H)^m / m!  psi,  H frozen at A[n] = A(t_n + dt/2)
 *                                                              north_star; Eq. (2) L138 midpoint (D1, D2, D7)
 *   rho(r) = sum_n f_n |psi_n(r)|^2 after every step           north_star; D13
 *   overlap S = dv * Phi^H Psi                                 PAPER.md L283 (CGEMM(1)), L132
 *
 * Layout: psi[dom][ix][iy][iz][n] complex128 (orbital index fastest, D12);
 * grid point index r = (ix*ny + iy)*nz + iz; beta[dom][r][p] complex128; D[dom][p];
 * vloc[dom][r]; occ[dom][n]; A[step][a_ndom][3] with a_ndom in {1, ndom} (D8).
 *
 * Parallelism: OpenMP over grid points only; reductions are summed in a fixed order so a
 * run is reproducible for a fixed thread count.  No blocking, fusion or reordering beyond
 * the definition above.
 *
 * Pins (tests/test_oracle_pins.py): plane-wave closed form, dense Kronecker H, dense
 * eigen-polynomial and expm on 16^3, Hermiticity, exact Taylor-4 norm identity, rank-1
 * projector closed form, Eq. (5) special case, density sum rule, batch independence,
 * Horner == term sum, brute force on an anisotropic 6x5x7 grid, 4th-order convergence.
 * mlmd_ref_propagate_split (the literal Eq. (2) step, end of this file) is pinned by
 * tests/test_oracle_split_pins.py: rank-1 kick closed form, reduction to the Taylor step, kick phase on
 * eigenvectors, dense Kronecker matrices, leading error term against expm.
 * Absolute values printed by the paper: none exist (the paper prints no psi/rho numbers).
 */
#include <complex.h>
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef double complex zc;

#define MLMD_REF_NO_KINETIC 1 /* oracle-internal switch for pin P6: drop -1/2 D2 - iA.D1 + 1/2|A|^2 */
#define MLMD_REF_HORNER 2     /* pin P10: evaluate the same polynomial in Horner form */
#define MLMD_REF_NO_LOCAL 4   /* split step (Eq. 2): drop the whole local part, out = V_NL u */
#define MLMD_REF_ORDER2 8     /* the paper's own local discretisation ("nearest-neighbor mesh points", L283
                               * "7-point star stencil"): 2nd-order central differences c2 = [1, -2, 1] / h^2,
                               * c1 = [-1/2, 0, 1/2] / h instead of north_star's 4th-order ones */

static const double C2[5] = {-1.0 / 12.0, 4.0 / 3.0, -5.0 / 2.0, 4.0 / 3.0, -1.0 / 12.0};
static const double C1[5] = {1.0 / 12.0, -2.0 / 3.0, 0.0, 2.0 / 3.0, -1.0 / 12.0};
/* 2nd order (7-point star), written on the same five offsets j = -2..2 */
static const double C2_O2[5] = {0.0, 1.0, -2.0, 1.0, 0.0};
static const double C1_O2[5] = {0.0, -0.5, 0.0, 0.5, 0.0};

static int wrap(int i, int n) {
    i %= n;
    return i < 0 ? i + n : i;
}

int mlmd_ref_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* out = H u for ONE domain.  u, out: [ngrid][norb]; beta: [ngrid][nproj]; D: [nproj]. */
int mlmd_ref_apply_h(int nx, int ny, int nz, double hx, double hy, double hz, int norb, int nproj,
                     const zc *u, zc *out, const double *vloc, const zc *beta, const double *D,
                     const double *A, int flags) {
    const int n3[3] = {nx, ny, nz};
    const double h[3] = {hx, hy, hz};
    const long ngrid = (long)nx * ny * nz;
    const double dv = hx * hy * hz;
    const double A2 = A[0] * A[0] + A[1] * A[1] + A[2] * A[2];
    const int kinetic = !(flags & MLMD_REF_NO_KINETIC);
    const double *c2 = (flags & MLMD_REF_ORDER2) ? C2_O2 : C2;
    const double *c1 = (flags & MLMD_REF_ORDER2) ? C1_O2 : C1;

    if (flags & MLMD_REF_NO_LOCAL) {
        for (size_t e = 0; e < (size_t)ngrid * norb; ++e) out[e] = 0.0;
    } else {
    /* local part: -1/2 D2 u - i A.D1 u + (V_loc + 1/2|A|^2) u */
#pragma omp parallel for collapse(2) schedule(static)
    for (int ix = 0; ix < nx; ++ix)
        for (int iy = 0; iy < ny; ++iy)
            for (int iz = 0; iz < nz; ++iz) {
                const int i3[3] = {ix, iy, iz};
                const long r = ((long)ix * ny + iy) * nz + iz;
                const double vr = vloc[r] + (kinetic ? 0.5 * A2 : 0.0);
                for (int n = 0; n < norb; ++n) out[r * norb + n] = vr * u[r * norb + n];
                if (!kinetic) continue;
                for (int d = 0; d < 3; ++d)
                    for (int j = -2; j <= 2; ++j) {
                        int q3[3] = {i3[0], i3[1], i3[2]};
                        q3[d] = wrap(i3[d] + j, n3[d]);
                        const long rr = ((long)q3[0] * ny + q3[1]) * nz + q3[2];
                        const zc coef = -0.5 * c2[j + 2] / (h[d] * h[d]) - I * A[d] * c1[j + 2] / h[d];
                        for (int n = 0; n < norb; ++n) out[r * norb + n] += coef * u[rr * norb + n];
                    }
            }
    }
    if (nproj <= 0) return 0;

    /* nonlocal part: C[p][n] = sum_r conj(beta[r][p]) u[r][n]; out[r][n] += sum_p beta[r][p] D_p dv C[p][n] */
    const int nt = mlmd_ref_num_threads();
    zc *part = (zc *)calloc((size_t)nt * nproj * norb, sizeof(zc));
    zc *C = (zc *)calloc((size_t)nproj * norb, sizeof(zc));
    if (!part || !C) {
        free(part);
        free(C);
        return 5;
    }
#pragma omp parallel num_threads(nt)
    {
#ifdef _OPENMP
        zc *mine = part + (size_t)omp_get_thread_num() * nproj * norb;
#else
        zc *mine = part;
#endif
#pragma omp for schedule(static)
        for (long r = 0; r < ngrid; ++r)
            for (int p = 0; p < nproj; ++p) {
                const zc b = conj(beta[r * nproj + p]);
                for (int n = 0; n < norb; ++n) mine[(size_t)p * norb + n] += b * u[r * norb + n];
            }
    }
    for (int t = 0; t < nt; ++t) /* fixed order */
        for (long k = 0; k < (long)nproj * norb; ++k) C[k] += part[(size_t)t * nproj * norb + k];
#pragma omp parallel for schedule(static)
    for (long r = 0; r < ngrid; ++r)
        for (int p = 0; p < nproj; ++p) {
            const zc bd = beta[r * nproj + p] * (D[p] * dv);
            for (int n = 0; n < norb; ++n) out[r * norb + n] += bd * C[(size_t)p * norb + n];
        }
    free(part);
    free(C);
    return 0;
}

/* rho[dom][r] = sum_n occ[dom][n] |psi[dom][r][n]|^2 */
int mlmd_ref_density(int ndom, long ngrid, int norb, const zc *psi, const double *occ, double *rho) {
    for (int dom = 0; dom < ndom; ++dom) {
        const zc *p = psi + (size_t)dom * ngrid * norb;
#pragma omp parallel for schedule(static)
        for (long r = 0; r < ngrid; ++r) {
            double s = 0.0;
            for (int n = 0; n < norb; ++n) {
                const zc v = p[r * norb + n];
                s += occ[(size_t)dom * norb + n] * (creal(v) * creal(v) + cimag(v) * cimag(v));
            }
            rho[(size_t)dom * ngrid + r] = s;
        }
    }
    return 0;
}

/* S[dom][m][n] = dv * sum_r conj(phi[dom][r][m]) psi[dom][r][n] */
int mlmd_ref_overlap(int ndom, long ngrid, int norb, double dv, const zc *phi, const zc *psi, zc *S) {
    for (int dom = 0; dom < ndom; ++dom) {
        const zc *a = phi + (size_t)dom * ngrid * norb;
        const zc *b = psi + (size_t)dom * ngrid * norb;
        zc *s = S + (size_t)dom * norb * norb;
#pragma omp parallel for schedule(static)
        for (int m = 0; m < norb; ++m)
            for (int n = 0; n < norb; ++n) {
                zc acc = 0.0;
                for (long r = 0; r < ngrid; ++r) acc += conj(a[r * norb + m]) * b[r * norb + n];
                s[(size_t)m * norb + n] = dv * acc;
            }
    }
    return 0;
}

/* nsteps Taylor-4 steps on every domain, in place; rho (may be NULL) from the last step. */
int mlmd_ref_propagate(int ndom, int nx, int ny, int nz, double hx, double hy, double hz, int norb,
                       int nproj, zc *psi, const double *occ, const double *vloc, const zc *beta,
                       const double *D, int nsteps, double dt, const double *A, int a_ndom,
                       double *rho, int flags) {
    const long ngrid = (long)nx * ny * nz;
    const size_t ne = (size_t)ngrid * norb;
    zc *phi = (zc *)malloc(ne * sizeof(zc));
    zc *hphi = (zc *)malloc(ne * sizeof(zc));
    zc *acc = (zc *)malloc(ne * sizeof(zc));
    if (!phi || !hphi || !acc) {
        free(phi);
        free(hphi);
        free(acc);
        return 5;
    }
    int rc = 0;
    for (int dom = 0; dom < ndom && !rc; ++dom) {
        zc *p = psi + (size_t)dom * ne;
        const double *v = vloc + (size_t)dom * ngrid;
        const zc *b = beta ? beta + (size_t)dom * ngrid * nproj : NULL;
        const double *d = D ? D + (size_t)dom * nproj : NULL;
        for (int step = 0; step < nsteps && !rc; ++step) {
            const double *Av = A + ((size_t)step * a_ndom + (a_ndom == 1 ? 0 : dom)) * 3;
            if (flags & MLMD_REF_HORNER) {
                /* w_4 = psi; w_{k-1} = psi + (-i dt/k) H w_k; psi_new = w_0 */
                memcpy(phi, p, ne * sizeof(zc));
                for (int k = 4; k >= 1 && !rc; --k) {
                    rc = mlmd_ref_apply_h(nx, ny, nz, hx, hy, hz, norb, nproj, phi, hphi, v, b, d, Av, flags);
                    const zc f = -I * dt / (double)k;
                    for (size_t e = 0; e < ne; ++e) phi[e] = p[e] + f * hphi[e];
                }
                memcpy(p, phi, ne * sizeof(zc));
            } else {
                /* phi_0 = psi; phi_m = (-i dt/m) H phi_{m-1}; psi_new = sum_{m=0..4} phi_m */
                memcpy(phi, p, ne * sizeof(zc));
                memcpy(acc, p, ne * sizeof(zc));
                for (int m = 1; m <= 4 && !rc; ++m) {
                    rc = mlmd_ref_apply_h(nx, ny, nz, hx, hy, hz, norb, nproj, phi, hphi, v, b, d, Av, flags);
                    const zc f = -I * dt / (double)m;
                    for (size_t e = 0; e < ne; ++e) {
                        phi[e] = f * hphi[e];
                        acc[e] += phi[e];
                    }
                }
                memcpy(p, acc, ne * sizeof(zc));
            }
            if (rho) mlmd_ref_density(1, ngrid, norb, p, occ + (size_t)dom * norb, rho + (size_t)dom * ngrid);
        }
        if (rho && nsteps == 0)
            mlmd_ref_density(1, ngrid, norb, p, occ + (size_t)dom * norb, rho + (size_t)dom * ngrid);
    }
    free(phi);
    free(hphi);
    free(acc);
    return rc;
}


/* ---- the paper's literal Eq. (2) step (readings D27, D28) ----
 *
 *   psi <- K  exp(-i dt h_loc(t_n + dt/2))  K  psi ,     K = (1 - i dt/2 v_nl) / || 1 - i dt/2 v_nl ||
 *                                                                   PAPER.md Eq. (2), Eq. (3)
 *   h_loc = 1/2 (-i grad + A)^2 + V_loc  (same finite differences as above),  v_nl = dv B diag(D) B^H;
 *   with B = Psi(0) and D_p = const this v_nl is the nonlocal correction of Eq. (5)
 *   (delta = -i dt/2 * D * dv).
 *   D27: the norm in K's denominator is taken on the state K acts on, orbital by orbital, so that
 *        each half-kick returns every orbital with the norm it came in with:
 *        K psi_n = (psi_n - i dt/2 v_nl psi_n) * ||psi_n|| / ||psi_n - i dt/2 v_nl psi_n||.
 *   D28: exp(-i dt h_loc) is the same 4th-order Taylor sum as the full-H step, applied to h_loc
 *        alone (the paper's own local solver is only named, L147; NEXT-3).
 * kick_only is a bit mask: 1 skips the local propagator (pin S3); 2 evaluates exp(-i dt h_loc) by the paper's own
 * block-diagonal split-operator solver on 2nd-order differences (reading D33) instead of the Taylor sum; 4 takes the
 * Taylor sum on the 2nd-order (7-point) differences of reading D32 instead of the 4th-order ones.
 */
/* ---- the paper's own local solver: block-diagonal split-operator (reading D33) ----
 *
 * PAPER.md L147 (A.5): exp(-i dt h_loc) is evaluated by "data-parallel local Hamiltonian-dynamics solvers that perform
 * uniform operations on nearest-neighbor mesh points: (1) a block-diagonal split-operator solver for electronic wave
 * functions [41]" (Richardson 1991); L283: "7-point star stencil (on which local computation is based)".  The paper
 * prints no formula; reading D33 restates the published space-splitting scheme on the operator of reading D32:
 *
 *   h_loc = sum_d T_d + V_loc + 1/2|A|^2,   (T_d u)_j = a_d u_j + b_d u_{j+1} + conj(b_d) u_{j-1}   (periodic in j),
 *   a_d = 1/h_d^2,  b_d = -1/(2 h_d^2) - i A_d/(2 h_d)        (-1/2 D2 - i A.D1 with 2nd-order central differences)
 *   T_d = E_d + O_d:  E_d couples the pairs (j, j+1) with j even, O_d those with j odd (the last pair wraps: n_d even);
 *   on its pair each is the 2 x 2 block [[a_d/2, b_d], [conj(b_d), a_d/2]], whose exponential is closed-form:
 *   exp(-i tau block) = e^{-i tau a_d/2} [[cos(tau|b|), -i u sin(tau|b|)], [-i conj(u) sin(tau|b|), cos(tau|b|)]], u = b/|b|
 *
 *   U_loc(dt) = P(dt/2)  S_x S_y S_z  P(dt/2),   S_d = e^{-i dt/2 E_d} e^{-i dt O_d} e^{-i dt/2 E_d},
 *   P(tau) = exp(-i tau (V_loc(r) + 1/2|A|^2))  (a phase per grid point).
 * Every factor is unitary (any dt), the product is symmetric (S_x, S_y, S_z act along different axes and commute), so
 * U_loc(-dt) U_loc(dt) = 1 and the error per step is O(dt^3).  Returns 2 if an axis has an odd number of points.
 * Pins: tests/test_oracle_richardson_pins.py (dense expm of every factor, E + O = the pinned 2nd-order operator,
 * unitarity for any dt, time reversal, order of convergence).
 */
static void pair_sweep(zc *p, int nx, int ny, int nz, int norb, int axis, int parity, double tau, double a, zc b) {
    const int n[3] = {nx, ny, nz};
    const long stride[3] = {(long)ny * nz * norb, (long)nz * norb, (long)norb};
    const double mb = cabs(b);
    const zc u = b / mb;
    const double c = cos(tau * mb), s = sin(tau * mb);
    const zc ph = cexp(-I * tau * a * 0.5);
    const int o1 = (axis + 1) % 3, o2 = (axis + 2) % 3;
    for (int j = parity; j < n[axis]; j += 2) {
        const int jn = (j + 1) % n[axis];
        for (int i1 = 0; i1 < n[o1]; ++i1)
            for (int i2 = 0; i2 < n[o2]; ++i2) {
                zc *q0 = p + j * stride[axis] + i1 * stride[o1] + i2 * stride[o2];
                zc *q1 = p + jn * stride[axis] + i1 * stride[o1] + i2 * stride[o2];
                for (int m = 0; m < norb; ++m) {
                    const zc v0 = q0[m], v1 = q1[m];
                    q0[m] = ph * (c * v0 - I * u * s * v1);
                    q1[m] = ph * (-I * conj(u) * s * v0 + c * v1);
                }
            }
    }
}

int mlmd_ref_local_richardson(int nx, int ny, int nz, double hx, double hy, double hz, int norb, zc *psi,
                              const double *vloc, const double *Av, double dt) {
    if (nx % 2 || ny % 2 || nz % 2) return 2;
    const long ngrid = (long)nx * ny * nz;
    const double hh[3] = {hx, hy, hz};
    const double a2 = 0.5 * (Av[0] * Av[0] + Av[1] * Av[1] + Av[2] * Av[2]);
    for (int half = 0; half < 2; ++half) {
        for (long r = 0; r < ngrid; ++r) {
            const zc f = cexp(-I * (0.5 * dt) * (vloc[r] + a2));
            for (int m = 0; m < norb; ++m) psi[r * norb + m] *= f;
        }
        if (half == 1) break;
        for (int d = 0; d < 3; ++d) {
            const double a = 1.0 / (hh[d] * hh[d]);
            const zc b = -0.5 / (hh[d] * hh[d]) - I * Av[d] / (2.0 * hh[d]);
            pair_sweep(psi, nx, ny, nz, norb, d, 0, 0.5 * dt, a, b);
            pair_sweep(psi, nx, ny, nz, norb, d, 1, dt, a, b);
            pair_sweep(psi, nx, ny, nz, norb, d, 0, 0.5 * dt, a, b);
        }
    }
    return 0;
}

static double col_norm2(const zc *u, long ngrid, int norb, int n) {
    double s = 0.0;
    for (long r = 0; r < ngrid; ++r) {
        const zc v = u[r * norb + n];
        s += creal(v) * creal(v) + cimag(v) * cimag(v);
    }
    return s;
}

static int half_kick(int nx, int ny, int nz, double hx, double hy, double hz, int norb, int nproj, zc *p,
                     zc *vp, const double *vloc, const zc *beta, const double *D, const double *Av, double dt) {
    const long ngrid = (long)nx * ny * nz;
    int rc = mlmd_ref_apply_h(nx, ny, nz, hx, hy, hz, norb, nproj, p, vp, vloc, beta, D, Av, MLMD_REF_NO_LOCAL);
    if (rc) return rc;
    for (int n = 0; n < norb; ++n) {
        const double before = col_norm2(p, ngrid, norb, n);
        for (long r = 0; r < ngrid; ++r) p[r * norb + n] -= I * (0.5 * dt) * vp[r * norb + n];
        const double after = col_norm2(p, ngrid, norb, n);
        const double s = after > 0.0 ? sqrt(before / after) : 1.0;
        for (long r = 0; r < ngrid; ++r) p[r * norb + n] *= s;
    }
    return 0;
}

int mlmd_ref_propagate_split(int ndom, int nx, int ny, int nz, double hx, double hy, double hz, int norb,
                             int nproj, zc *psi, const double *occ, const double *vloc, const zc *beta,
                             const double *D, int nsteps, double dt, const double *A, int a_ndom,
                             double *rho, int kick_only) {
    const long ngrid = (long)nx * ny * nz;
    const size_t ne = (size_t)ngrid * norb;
    zc *phi = (zc *)malloc(ne * sizeof(zc));
    zc *hphi = (zc *)malloc(ne * sizeof(zc));
    zc *acc = (zc *)malloc(ne * sizeof(zc));
    if (!phi || !hphi || !acc) {
        free(phi);
        free(hphi);
        free(acc);
        return 5;
    }
    int rc = 0;
    for (int dom = 0; dom < ndom && !rc; ++dom) {
        zc *p = psi + (size_t)dom * ne;
        const double *v = vloc + (size_t)dom * ngrid;
        const zc *b = beta ? beta + (size_t)dom * ngrid * nproj : NULL;
        const double *d = D ? D + (size_t)dom * nproj : NULL;
        for (int step = 0; step < nsteps && !rc; ++step) {
            const double *Av = A + ((size_t)step * a_ndom + (a_ndom == 1 ? 0 : dom)) * 3;
            if (nproj > 0) rc = half_kick(nx, ny, nz, hx, hy, hz, norb, nproj, p, hphi, v, b, d, Av, dt);
            if (!(kick_only & 1) && (kick_only & 2) && !rc) {
                /* reading D33: the paper's own local solver (block-diagonal split-operator, 2nd-order differences) */
                rc = mlmd_ref_local_richardson(nx, ny, nz, hx, hy, hz, norb, p, v, Av, dt);
            } else if (!(kick_only & 1) && !rc) {
                /* phi_0 = psi; phi_m = (-i dt/m) h_loc phi_{m-1}; psi_new = sum_{m=0..4} phi_m */
                memcpy(phi, p, ne * sizeof(zc));
                memcpy(acc, p, ne * sizeof(zc));
                for (int m = 1; m <= 4 && !rc; ++m) {
                    rc = mlmd_ref_apply_h(nx, ny, nz, hx, hy, hz, norb, 0, phi, hphi, v, NULL, NULL, Av,
                                          (kick_only & 4) ? MLMD_REF_ORDER2 : 0);
                    const zc f = -I * dt / (double)m;
                    for (size_t e = 0; e < ne; ++e) {
                        phi[e] = f * hphi[e];
                        acc[e] += phi[e];
                    }
                }
                memcpy(p, acc, ne * sizeof(zc));
            }
            if (nproj > 0 && !rc) rc = half_kick(nx, ny, nz, hx, hy, hz, norb, nproj, p, hphi, v, b, d, Av, dt);
            if (rho) mlmd_ref_density(1, ngrid, norb, p, occ + (size_t)dom * norb, rho + (size_t)dom * ngrid);
        }
        if (rho && nsteps == 0)
            mlmd_ref_density(1, ngrid, norb, p, occ + (size_t)dom * norb, rho + (size_t)dom * ngrid);
    }
    free(phi);
    free(hphi);
    free(acc);
    return rc;
}

/* Occupations of the reference orbitals and number of excited electrons (LFD returns the
 * occupation numbers f_s to QXMD; L159: n_exc per domain "is computed from f_s"; L283: from the overlap
 * matrix between the orbitals at time t and 0).  The paper gives no formula; reading D29:
 *   f_s(t)  = sum_n f_n |S_sn|^2 ,  S_sn = <psi_s(0)|psi_n(t)>   (orbital n carries f_n electrons)
 *   n_exc   = sum_s max(f_s(0) - f_s(t), 0)                      (electrons that left their t=0 orbitals)
 * S: [ndom][norb][norb] as mlmd_ref_overlap(phi = Psi(0), psi = Psi(t)) writes it; occ: [ndom][norb]. */
int mlmd_ref_occupations(int ndom, int norb, const zc *S, const double *occ, double *f, double *nexc) {
    for (int dom = 0; dom < ndom; ++dom) {
        double holes = 0.0;
        for (int s = 0; s < norb; ++s) {
            double acc = 0.0;
            for (int n = 0; n < norb; ++n) {
                const zc v = S[((size_t)dom * norb + s) * norb + n];
                acc += occ[(size_t)dom * norb + n] * (creal(v) * creal(v) + cimag(v) * cimag(v));
            }
            f[(size_t)dom * norb + s] = acc;
            const double lost = occ[(size_t)dom * norb + s] - acc;
            if (lost > 0.0) holes += lost;
        }
        nexc[dom] = holes;
    }
    return 0;
}

/* ---- observables of SURVEY.md 8(f) NEXT-2 ("GEMMification is applied to nonlocal correction in
 * energy and electric current ... with the latter used in Maxwell's equations") ----
 *
 * Nonlocal energy of one domain:  E_nl = sum_n f_n <psi_n|V_NL|psi_n>,  V_NL = dv B diag(D) B^H, <a|b> = dv sum conj(a) b
 *                                      = dv^2 sum_n f_n sum_p D_p |sum_r conj(beta[r][p]) psi[r][n]|^2 .            */
int mlmd_ref_energy_nl(int ndom, long ngrid, int norb, int nproj, double dv, const zc *psi, const double *occ,
                       const zc *beta, const double *D, double *E) {
    for (int dom = 0; dom < ndom; ++dom) {
        const zc *p = psi + (size_t)dom * ngrid * norb;
        const zc *b = beta + (size_t)dom * ngrid * nproj;
        double *en = (double *)calloc((size_t)norb, sizeof(double));   /* one orbital per thread, summed in order below */
        if (!en) return 5;
#pragma omp parallel for schedule(dynamic)
        for (int n = 0; n < norb; ++n)
            for (int q = 0; q < nproj; ++q) {
                zc c = 0.0;
                for (long r = 0; r < ngrid; ++r) c += conj(b[r * nproj + q]) * p[r * norb + n];
                en[n] += occ[(size_t)dom * norb + n] * D[(size_t)dom * nproj + q] * dv * dv * (creal(c) * creal(c) + cimag(c) * cimag(c));
            }
        double e = 0.0;
        for (int n = 0; n < norb; ++n) e += en[n];
        free(en);
        E[dom] = e;
    }
    return 0;
}

/* Local current of one domain (the velocity operator of h_loc in Eq. (3) L142 is -i grad + A; reading D30: the
 * nonlocal-pseudopotential term -i[r, V_NL] of the TDCDFT current is named at L201 but not given and is left out):
 *   J_d = sum_n f_n Re <psi_n| -i D1_d + A_d |psi_n>,   D1_d = the 4th-order central first difference of H.
 * A: [a_ndom][3]; J: [ndom][3]. */
int mlmd_ref_current(int ndom, int nx, int ny, int nz, double hx, double hy, double hz, int norb, const zc *psi,
                     const double *occ, const double *A, int a_ndom, double *J, int flags /* MLMD_REF_ORDER2: 2nd-order D1 */) {
    const double *c1 = (flags & MLMD_REF_ORDER2) ? C1_O2 : C1;
    const int n3[3] = {nx, ny, nz};
    const double h[3] = {hx, hy, hz};
    const long ngrid = (long)nx * ny * nz;
    const double dv = hx * hy * hz;
    for (int dom = 0; dom < ndom; ++dom) {
        const zc *p = psi + (size_t)dom * ngrid * norb;
        const double *Av = A + (size_t)(a_ndom == 1 ? 0 : dom) * 3;
        for (int d = 0; d < 3; ++d) {
            double *plane = (double *)calloc((size_t)nx, sizeof(double));   /* one x-plane per thread, summed in order below */
            if (!plane) return 5;
#pragma omp parallel for schedule(static)
            for (int ix = 0; ix < nx; ++ix) {
                double acc = 0.0;
                for (int iy = 0; iy < ny; ++iy)
                    for (int iz = 0; iz < nz; ++iz) {
                        const int i3[3] = {ix, iy, iz};
                        const long r = ((long)ix * ny + iy) * nz + iz;
                        for (int n = 0; n < norb; ++n) {
                            zc g = 0.0;
                            for (int j = -2; j <= 2; ++j) {
                                int q3[3] = {i3[0], i3[1], i3[2]};
                                q3[d] = wrap(i3[d] + j, n3[d]);
                                const long rr = ((long)q3[0] * ny + q3[1]) * nz + q3[2];
                                g += c1[j + 2] / h[d] * p[rr * norb + n];
                            }
                            const zc u = p[r * norb + n];
                            acc += occ[(size_t)dom * norb + n] * dv * creal(conj(u) * (-I * g + Av[d] * u));
                        }
                    }
                plane[ix] = acc;
            }
            double acc = 0.0;
            for (int ix = 0; ix < nx; ++ix) acc += plane[ix];
            free(plane);
            J[(size_t)dom * 3 + d] = acc;
        }
    }
    return 0;
}

/* Nonlocal (pseudopotential) part of the TDCDFT current of one batch ("GEMMification is applied to
 * nonlocal correction in energy and electric current (TDCDFT), with the latter used in Maxwell's equations"; the paper
 * prints no formula: reading D31 in DESIGN.md).  The velocity operator of a nonlocal potential is -i [r, V_NL]; with
 * V_NL = dv sum_p |beta_p> D_p <beta_p| its expectation value is
 *   J_d = sum_n f_n <psi_n| -i [r_d, V_NL] |psi_n> = 2 dv^2 sum_n f_n sum_p D_p Im( conj(G_dpn) C_pn ),
 *   C_pn = sum_r conj(beta_p(r)) psi_n(r),   G_dpn = sum_r conj(rbeta_dp(r)) psi_n(r),   rbeta_dp(r) = (r - R_p)_d beta_p(r)
 * ((r - R_p): position relative to the projector's centre, minimum image; a constant shift R_p commutes, so each term
 * is the commutator with r itself).  The caller supplies the three arrays rbeta_d: [ndom][ngrid][nproj] each.
 * J: [ndom][3]. */
int mlmd_ref_current_nl(int ndom, long ngrid, int norb, int nproj, double dv, const zc *psi, const double *occ,
                        const zc *beta, const zc *rbeta /* [3][ndom][ngrid][nproj] */, const double *D, double *J) {
    for (int dom = 0; dom < ndom; ++dom) {
        const zc *p = psi + (size_t)dom * ngrid * norb;
        const zc *b = beta + (size_t)dom * ngrid * nproj;
        zc *C = (zc *)calloc((size_t)nproj * norb, sizeof(zc));
        zc *G = (zc *)calloc((size_t)nproj * norb, sizeof(zc));
        if (!C || !G) {
            free(C);
            free(G);
            return 5;
        }
        for (long r = 0; r < ngrid; ++r)
            for (int q = 0; q < nproj; ++q)
                for (int n = 0; n < norb; ++n) C[(size_t)q * norb + n] += conj(b[r * nproj + q]) * p[r * norb + n];
        for (int d = 0; d < 3; ++d) {
            const zc *rb = rbeta + ((size_t)d * ndom + dom) * ngrid * nproj;
            memset(G, 0, (size_t)nproj * norb * sizeof(zc));
            for (long r = 0; r < ngrid; ++r)
                for (int q = 0; q < nproj; ++q)
                    for (int n = 0; n < norb; ++n) G[(size_t)q * norb + n] += conj(rb[r * nproj + q]) * p[r * norb + n];
            double acc = 0.0;
            for (int n = 0; n < norb; ++n)
                for (int q = 0; q < nproj; ++q)
                    acc += occ[(size_t)dom * norb + n] * D[(size_t)dom * nproj + q] *
                           cimag(conj(G[(size_t)q * norb + n]) * C[(size_t)q * norb + n]);
            J[(size_t)dom * 3 + d] = 2.0 * dv * dv * acc;
        }
        free(C);
        free(G);
    }
    return 0;
}

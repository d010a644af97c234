/*
 * u1u1_oracle.c -- fp64 CPU ORACLE for the U(1)xU(1) leapfrog hot path.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may load it.  It shares no code,
 * header, table or helper with the CUDA path (paper_2208_01525_b200/csrc); the CUDA path
 * never calls it.
 *
 * What it is: a plain, slow, obviously-correct restatement of the discretised equations of
 * Correia & Martins, arXiv:2208.01525, step by step in the paper's order:
 *   Pi,Psi kick (Eq. 17-18)  ->  E,H kick (:137-143, Eq. 20-21)
 *   -> drift (:149-158, Eq. 23-26), with delta (:133, Eq. 19), omega (:147, Eq. 22) and the
 *   a^{2 beta} factor of Eq. 12-16 (:87-105).  Diagnostics: Gauss laws (:73-77, Eq. 9-10),
 *   windings / pierced cells (:183-194, :234, :252), Lagrangian and velocity densities
 *   (:196-200 Eq. 33, :214-224 Eq. 36-37).
 * Readings of garbled / silent passages are those of DESIGN.md section 3 (R-1 .. R-19).
 *
 * No blocking, fusion or reordering: every function is a triple loop over sites that
 * evaluates the printed formula.  All arithmetic is double precision.
 *
 * State layout ("canonical"): double state[20][nz][ny][nx], x fastest, components
 *   0 phi_re 1 phi_im 2 Pi_re 3 Pi_im 4 psi_re 5 psi_im 6 Psi_re 7 Psi_im
 *   8..10 thetaA_{x,y,z}  11..13 E_{x,y,z}  14..16 thetaB_{x,y,z}  17..19 H_{x,y,z}
 * with theta_i = dx * A_i (link phase, NON-compact: never wrapped) and E_i = dA_i/dtau.
 *
 * Pins (tests/test_oracle_pins.py): energy conservation, one-step Gauss identity, gauge
 * covariance, static vortex + Bogomolny tension 2 pi sigma^2, sector symmetry
 * (:79), brute-force windings and the "cell value 2" statement (:252), kappa=0 decoupling,
 * homogeneous-mode ODE, Philox known-answer vectors.
 * Cooling (O-12, Eq. 27-30): monotone energy decrease, relaxed vortex as a fixed point, equivalence with
 *   kick+drift from zero momenta when kappa = 0.
 * Diagnostic combinations (tests/test_oracle_pins_diag.py): the densities of orc_densities through the variational
 *   principle (their weighted sum's gradient is the pinned kicks' right-hand side), virial theorems, the Bogomolny
 *   vortex; V_int on hand-computed sites; the near-cut mask of orc_windings on hand-built links.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#ifndef M_PI
#define M_PI 3.14159265358979323846
#endif

typedef struct {
    int nx, ny, nz;
    double dx;
} orc_lattice;

typedef struct {
    double lambda1, lambda2; /* lambda_p0, lambda_q0  (PAPER.md:52 Eq. 4, :89 Eq. 12) */
    double e1, e2;           /* e_p0, e_q0 */
    double eta1, eta2;       /* sigma_p, sigma_q (the VEVs; BASELINE.json calls them eta) */
    double kappa;            /* kappa_0 */
} orc_couplings;

enum { PHI = 0, PIM = 2, PSI = 4, PSM = 6, THA = 8, EA = 11, THB = 14, HB = 17 };

static size_t vol(const orc_lattice *L) { return (size_t)L->nx * L->ny * L->nz; }

static size_t site(const orc_lattice *L, int ix, int iy, int iz)
{
    ix = ((ix % L->nx) + L->nx) % L->nx; /* periodic in all three directions */
    iy = ((iy % L->ny) + L->ny) % L->ny;
    iz = ((iz % L->nz) + L->nz) % L->nz;
    return (size_t)ix + (size_t)L->nx * ((size_t)iy + (size_t)L->ny * (size_t)iz);
}

/* site displaced by `n` steps along direction dir (0=x,1=y,2=z) */
static size_t shift(const orc_lattice *L, int ix, int iy, int iz, int dir, int n)
{
    return site(L, ix + (dir == 0 ? n : 0), iy + (dir == 1 ? n : 0), iz + (dir == 2 ? n : 0));
}

/* ------------------------------------------------------------------------------------------
 * O-3  per-step scalars.  PAPER.md:133 Eq. 19 (alpha = 2, :135), :147 Eq. 22, :89 Eq. 12.
 *   a ∝ t^m  <=>  a ∝ tau^p with p = m/(1-m); normalised a(tau_norm) = 1 (reading R-3).
 *   out = { a, c = a^{2 beta}, delta, omega }
 * ---------------------------------------------------------------------------------------- */
void orc_scalars(double tau, double m, double beta, double dtau, double tau_norm, double out[4])
{
    const double alpha = 2.0;
    double p = m / (1.0 - m);
    double a = (m == 0.0) ? 1.0 : pow(tau / tau_norm, p);
    double c = pow(a, 2.0 * beta);
    double delta = (m == 0.0) ? 0.0 : 0.5 * alpha * (m * dtau) / ((1.0 - m) * tau);
    double omega = delta * (1.0 - beta);
    out[0] = a;
    out[1] = c;
    out[2] = delta;
    out[3] = omega;
}

/* O-1  forward hop U_i(x) f(x+i), U = exp(-i theta)  (D = d - iA, Eq. 2, R-2) */
static void hop_forward(const orc_lattice *L, const double *f_re, const double *f_im,
                        const double *theta_dir, int ix, int iy, int iz, int dir, double *re,
                        double *im)
{
    size_t x = site(L, ix, iy, iz), xp = shift(L, ix, iy, iz, dir, +1);
    double cs = cos(theta_dir[x]), sn = sin(theta_dir[x]);
    /* (cs - i sn)(a + i b) */
    *re = cs * f_re[xp] + sn * f_im[xp];
    *im = cs * f_im[xp] - sn * f_re[xp];
}

/* O-1  backward hop conj(U_i(x-i)) f(x-i) */
static void hop_backward(const orc_lattice *L, const double *f_re, const double *f_im,
                         const double *theta_dir, int ix, int iy, int iz, int dir, double *re,
                         double *im)
{
    size_t xm = shift(L, ix, iy, iz, dir, -1);
    double cs = cos(theta_dir[xm]), sn = sin(theta_dir[xm]);
    /* (cs + i sn)(a + i b) */
    *re = cs * f_re[xm] - sn * f_im[xm];
    *im = cs * f_im[xm] + sn * f_re[xm];
}

/* O-2  plaquette P_ij(x) = theta_i(x) + theta_j(x+i) - theta_i(x+j) - theta_j(x) = dx^2 F_ij */
static double plaquette(const orc_lattice *L, const double *theta /* 3 planes */, int ix, int iy,
                        int iz, int i, int j)
{
    size_t V = vol(L);
    const double *ti = theta + (size_t)i * V, *tj = theta + (size_t)j * V;
    return ti[site(L, ix, iy, iz)] + tj[shift(L, ix, iy, iz, i, +1)] -
           ti[shift(L, ix, iy, iz, j, +1)] - tj[site(L, ix, iy, iz)];
}

/* ------------------------------------------------------------------------------------------
 * O-4a  scalar momentum kick, one sector.  PAPER.md:110 (Eq. 17, first intact line) and
 * :126-129 (Eq. 18):
 *   (1+delta) Pi+ = (1-delta) Pi- + dtau [ D-_j D+_j phi
 *                     - c phi ( lambda/2 (|phi|^2 - sigma^2) - kappa (|other|^2 - sigma_o^2) ) ]
 * All right-hand sides at time tau.  Reads positions only -> in-place on the momentum.
 * ---------------------------------------------------------------------------------------- */
static void kick_scalar_sector(const orc_lattice *L, const double *f_re, const double *f_im,
                               const double *o_re, const double *o_im, const double *theta,
                               double *mom_re, double *mom_im, double lambda, double sigma,
                               double sigma_o, double kappa, double c, double delta, double dtau)
{
    size_t V = vol(L);
    double dx2 = L->dx * L->dx;
    int iz;
#pragma omp parallel for
    for (iz = 0; iz < L->nz; iz++)
        for (int iy = 0; iy < L->ny; iy++)
            for (int ix = 0; ix < L->nx; ix++) {
                size_t x = site(L, ix, iy, iz);
                double lap_re = 0.0, lap_im = 0.0;
                for (int j = 0; j < 3; j++) {
                    double fr, fi, br, bi;
                    hop_forward(L, f_re, f_im, theta + (size_t)j * V, ix, iy, iz, j, &fr, &fi);
                    hop_backward(L, f_re, f_im, theta + (size_t)j * V, ix, iy, iz, j, &br, &bi);
                    lap_re += (fr + br - 2.0 * f_re[x]) / dx2;
                    lap_im += (fi + bi - 2.0 * f_im[x]) / dx2;
                }
                double mod2 = f_re[x] * f_re[x] + f_im[x] * f_im[x];
                double omod2 = o_re[x] * o_re[x] + o_im[x] * o_im[x];
                double bracket = 0.5 * lambda * (mod2 - sigma * sigma) -
                                 kappa * (omod2 - sigma_o * sigma_o);
                double rhs_re = lap_re - c * f_re[x] * bracket;
                double rhs_im = lap_im - c * f_im[x] * bracket;
                mom_re[x] = ((1.0 - delta) * mom_re[x] + dtau * rhs_re) / (1.0 + delta);
                mom_im[x] = ((1.0 - delta) * mom_im[x] + dtau * rhs_im) / (1.0 + delta);
            }
}

void orc_kick_scalars(const orc_lattice *L, const orc_couplings *K, double *state, double c,
                      double delta, double dtau)
{
    size_t V = vol(L);
    double *s = state;
    kick_scalar_sector(L, s + PHI * V, s + (PHI + 1) * V, s + PSI * V, s + (PSI + 1) * V,
                       s + THA * V, s + PIM * V, s + (PIM + 1) * V, K->lambda1, K->eta1, K->eta2,
                       K->kappa, c, delta, dtau);
    kick_scalar_sector(L, s + PSI * V, s + (PSI + 1) * V, s + PHI * V, s + (PHI + 1) * V,
                       s + THB * V, s + PSM * V, s + (PSM + 1) * V, K->lambda2, K->eta2, K->eta1,
                       K->kappa, c, delta, dtau);
}

/* ------------------------------------------------------------------------------------------
 * O-4b  gauge momentum kick, one sector.  PAPER.md:139 Eq. 20 (readings R-4, R-6):
 *   (1+omega) E_i+ = (1-omega) E_i- + dtau [ - sum_{j!=i} d-_j F_ij + 2 e0^2 c Im(phi* D+_i phi) ]
 *   d-_j F_ij (x) = [P_ij(x) - P_ij(x-j)] / dx^3 ,   D+_i phi = (U_i phi(x+i) - phi(x)) / dx
 * ---------------------------------------------------------------------------------------- */
static void kick_gauge_sector(const orc_lattice *L, const double *f_re, const double *f_im,
                              const double *theta, double *E, double e0, double c, double omega,
                              double dtau)
{
    size_t V = vol(L);
    double dx = L->dx;
    int iz;
#pragma omp parallel for
    for (iz = 0; iz < L->nz; iz++)
        for (int iy = 0; iy < L->ny; iy++)
            for (int ix = 0; ix < L->nx; ix++) {
                size_t x = site(L, ix, iy, iz);
                for (int i = 0; i < 3; i++) {
                    double curl = 0.0;
                    for (int j = 0; j < 3; j++) {
                        if (j == i) continue;
                        int jx = ix - (j == 0), jy = iy - (j == 1), jz = iz - (j == 2);
                        curl += (plaquette(L, theta, ix, iy, iz, i, j) -
                                 plaquette(L, theta, jx, jy, jz, i, j)) /
                                (dx * dx * dx);
                    }
                    double hr, hi;
                    hop_forward(L, f_re, f_im, theta + (size_t)i * V, ix, iy, iz, i, &hr, &hi);
                    double Dre = (hr - f_re[x]) / dx, Dim = (hi - f_im[x]) / dx;
                    double current = f_re[x] * Dim - f_im[x] * Dre; /* Im(conj(phi) D+ phi) */
                    double rhs = -curl + 2.0 * e0 * e0 * c * current;
                    double *Ei = E + (size_t)i * V;
                    Ei[x] = ((1.0 - omega) * Ei[x] + dtau * rhs) / (1.0 + omega);
                }
            }
}

void orc_kick_gauge(const orc_lattice *L, const orc_couplings *K, double *state, double c,
                    double omega, double dtau)
{
    size_t V = vol(L);
    double *s = state;
    kick_gauge_sector(L, s + PHI * V, s + (PHI + 1) * V, s + THA * V, s + EA * V, K->e1, c, omega,
                      dtau);
    kick_gauge_sector(L, s + PSI * V, s + (PSI + 1) * V, s + THB * V, s + HB * V, K->e2, c, omega,
                      dtau);
}

/* O-5  friction of the damping prephase (BASELINE.json configs 2 and 5; reading R-11):
 * all four momenta are multiplied by f after the kick. */
void orc_friction(const orc_lattice *L, double *state, double f)
{
    size_t V = vol(L);
    static const int mom[10] = {2, 3, 6, 7, 11, 12, 13, 17, 18, 19};
    for (int k = 0; k < 10; k++)
        for (size_t x = 0; x < V; x++) state[(size_t)mom[k] * V + x] *= f;
}

/* O-6  drift.  PAPER.md:151-158 Eq. 23-26: phi += dtau Pi, psi += dtau Psi, A_i += dtau E_i,
 * B_i += dtau H_i   (theta = dx A  =>  theta_i += dtau dx E_i). */
void orc_drift(const orc_lattice *L, double *state, double dtau)
{
    size_t V = vol(L);
    for (size_t x = 0; x < V; x++) {
        for (int r = 0; r < 2; r++) {
            state[(PHI + r) * V + x] += dtau * state[(PIM + r) * V + x];
            state[(PSI + r) * V + x] += dtau * state[(PSM + r) * V + x];
        }
        for (int i = 0; i < 3; i++) {
            state[(THA + i) * V + x] += dtau * L->dx * state[(EA + i) * V + x];
            state[(THB + i) * V + x] += dtau * L->dx * state[(HB + i) * V + x];
        }
    }
}

/* One full timestep in the paper's order (PAPER.md:108 "executed first", :137 "Next",
 * :149 "To finish").  Positions at tau, momenta at tau - dtau/2 on entry. */
void orc_step(const orc_lattice *L, const orc_couplings *K, double *state, double tau, double m,
              double beta, double dtau, double tau_norm, double friction)
{
    double sc[4];
    orc_scalars(tau, m, beta, dtau, tau_norm, sc);
    orc_kick_scalars(L, K, state, sc[1], sc[2], dtau);
    orc_kick_gauge(L, K, state, sc[1], sc[3], dtau);
    if (friction != 1.0) orc_friction(L, state, friction);
    orc_drift(L, state, dtau);
}

/* ------------------------------------------------------------------------------------------
 * O-12  diffusive cooling, one explicit Euler step.  PAPER.md:164-177 Eq. 27-30 (readings R-8, R-20):
 *   d phi / d eta = D-_j D+_j phi - lambda_p0/2 (|phi|^2 - sigma_p^2) phi          (Eq. 27, no kappa term)
 *   d A_i / d eta = - sum_{j != i} d-_j F_ij + 2 e_p0^2 Im(phi* D+_i phi)          (Eq. 28, R-20)
 * and the mirror for (psi, B) (Eq. 29-30).  All right-hand sides are evaluated on the fields at eta
 * (into scratch arrays), then every field is advanced by dcool times its right-hand side.  No scale
 * factor, no momenta: on exit the momenta hold zero.  scratch = 10 * volume doubles.
 * ---------------------------------------------------------------------------------------- */
void orc_cool_step(const orc_lattice *L, const orc_couplings *K, double *state, double dcool,
                   double *scratch)
{
    size_t V = vol(L);
    double dx = L->dx, dx2 = dx * dx;
    for (int sec = 0; sec < 2; sec++) {
        const double *f_re = state + (sec ? PSI : PHI) * V, *f_im = f_re + V;
        const double *theta = state + (sec ? THB : THA) * V;
        double lambda = sec ? K->lambda2 : K->lambda1, sigma = sec ? K->eta2 : K->eta1;
        double e0 = sec ? K->e2 : K->e1;
        double *r_re = scratch + (size_t)(5 * sec) * V, *r_im = r_re + V, *r_A = r_im + V;
        for (int iz = 0; iz < L->nz; iz++)
            for (int iy = 0; iy < L->ny; iy++)
                for (int ix = 0; ix < L->nx; ix++) {
                    size_t x = site(L, ix, iy, iz);
                    double lap_re = 0.0, lap_im = 0.0;
                    for (int j = 0; j < 3; j++) {
                        double fr, fi, br, bi;
                        hop_forward(L, f_re, f_im, theta + (size_t)j * V, ix, iy, iz, j, &fr, &fi);
                        hop_backward(L, f_re, f_im, theta + (size_t)j * V, ix, iy, iz, j, &br, &bi);
                        lap_re += (fr + br - 2.0 * f_re[x]) / dx2;
                        lap_im += (fi + bi - 2.0 * f_im[x]) / dx2;
                    }
                    double mod2 = f_re[x] * f_re[x] + f_im[x] * f_im[x];
                    double pot = 0.5 * lambda * (mod2 - sigma * sigma);
                    r_re[x] = lap_re - pot * f_re[x];
                    r_im[x] = lap_im - pot * f_im[x];
                    for (int i = 0; i < 3; i++) {
                        double curl = 0.0;
                        for (int j = 0; j < 3; j++) {
                            if (j == i) continue;
                            int jx = ix - (j == 0), jy = iy - (j == 1), jz = iz - (j == 2);
                            curl += (plaquette(L, theta, ix, iy, iz, i, j) -
                                     plaquette(L, theta, jx, jy, jz, i, j)) / (dx * dx * dx);
                        }
                        double hr, hi;
                        hop_forward(L, f_re, f_im, theta + (size_t)i * V, ix, iy, iz, i, &hr, &hi);
                        double Dre = (hr - f_re[x]) / dx, Dim = (hi - f_im[x]) / dx;
                        r_A[(size_t)i * V + x] = -curl + 2.0 * e0 * e0 * (f_re[x] * Dim - f_im[x] * Dre);
                    }
                }
    }
    for (int sec = 0; sec < 2; sec++) {
        double *f_re = state + (sec ? PSI : PHI) * V, *f_im = f_re + V;
        double *theta = state + (sec ? THB : THA) * V;
        const double *r_re = scratch + (size_t)(5 * sec) * V, *r_im = r_re + V, *r_A = r_im + V;
        for (size_t x = 0; x < V; x++) {
            f_re[x] += dcool * r_re[x];
            f_im[x] += dcool * r_im[x];
            for (int i = 0; i < 3; i++) theta[(size_t)i * V + x] += dcool * dx * r_A[(size_t)i * V + x];
        }
    }
    static const int mom[10] = {2, 3, 6, 7, 11, 12, 13, 17, 18, 19};
    for (int k = 0; k < 10; k++) memset(state + (size_t)mom[k] * V, 0, V * sizeof(double));
}

/* ------------------------------------------------------------------------------------------
 * O-7  Gauss residual per site and sector.  PAPER.md:75-77 Eq. 9-10 (reading R-5):
 *   g(x) = sum_i [E_i(x) - E_i(x-i)]/dx - 2 e0^2 cG Im(conj(phi) Pi)
 * writes g, rho = 2 e0^2 cG Im(conj(phi) Pi), divE for sector `sec` (0 = p, 1 = q).
 * ---------------------------------------------------------------------------------------- */
void orc_gauss_field(const orc_lattice *L, const orc_couplings *K, const double *state, int sec,
                     double cG, double *g, double *rho, double *divE)
{
    size_t V = vol(L);
    const double *f_re = state + (sec ? PSI : PHI) * V, *f_im = f_re + V;
    const double *m_re = state + (sec ? PSM : PIM) * V, *m_im = m_re + V;
    const double *E = state + (sec ? HB : EA) * V;
    double e0 = sec ? K->e2 : K->e1;
    for (int iz = 0; iz < L->nz; iz++)
        for (int iy = 0; iy < L->ny; iy++)
            for (int ix = 0; ix < L->nx; ix++) {
                size_t x = site(L, ix, iy, iz);
                double d = 0.0;
                for (int i = 0; i < 3; i++)
                    d += (E[(size_t)i * V + x] - E[(size_t)i * V + shift(L, ix, iy, iz, i, -1)]) /
                         L->dx;
                double r = 2.0 * e0 * e0 * cG * (f_re[x] * m_im[x] - f_im[x] * m_re[x]);
                divE[x] = d;
                rho[x] = r;
                g[x] = d - r;
            }
}

/* ------------------------------------------------------------------------------------------
 * O-8  windings.  PAPER.md:183-188 ("sum of non-zero plaquettes"), construction per R-12:
 *   chi_i(x) = arg( conj(phi(x)) U_i(x) phi(x+i) )  in (-pi, pi],  atan2(0,0) = 0
 *   W_ij(x)  = round( [chi_i(x) + chi_j(x+i) - chi_i(x+j) - chi_j(x) + P_ij(x)] / 2 pi )
 * orientation index o: 0 = xy, 1 = yz, 2 = zx.  near[o][x] = 1 if any of the 4 link angles of
 * that plaquette has pi - |chi| < cut_tol (reading R-15).
 * ---------------------------------------------------------------------------------------- */
static double link_angle(const orc_lattice *L, const double *f_re, const double *f_im,
                         const double *theta, int ix, int iy, int iz, int dir)
{
    size_t V = vol(L), x = site(L, ix, iy, iz);
    double hr, hi;
    hop_forward(L, f_re, f_im, theta + (size_t)dir * V, ix, iy, iz, dir, &hr, &hi);
    double re = f_re[x] * hr + f_im[x] * hi; /* conj(phi) * hop */
    double im = f_re[x] * hi - f_im[x] * hr;
    if (re == 0.0 && im == 0.0) return 0.0;
    return atan2(im, re);
}

void orc_windings(const orc_lattice *L, const double *state, int sec, double cut_tol, int32_t *W,
                  uint8_t *near)
{
    size_t V = vol(L);
    const double *f_re = state + (sec ? PSI : PHI) * V, *f_im = f_re + V;
    const double *theta = state + (sec ? THB : THA) * V;
    static const int oi[3] = {0, 1, 2}, oj[3] = {1, 2, 0};
    for (int o = 0; o < 3; o++) {
        int i = oi[o], j = oj[o];
        for (int iz = 0; iz < L->nz; iz++)
            for (int iy = 0; iy < L->ny; iy++)
                for (int ix = 0; ix < L->nx; ix++) {
                    int xi = ix + (i == 0), yi = iy + (i == 1), zi = iz + (i == 2); /* x+i */
                    int xj = ix + (j == 0), yj = iy + (j == 1), zj = iz + (j == 2); /* x+j */
                    double c1 = link_angle(L, f_re, f_im, theta, ix, iy, iz, i);
                    double c2 = link_angle(L, f_re, f_im, theta, xi, yi, zi, j);
                    double c3 = link_angle(L, f_re, f_im, theta, xj, yj, zj, i);
                    double c4 = link_angle(L, f_re, f_im, theta, ix, iy, iz, j);
                    double sum = c1 + c2 - c3 - c4 + plaquette(L, theta, ix, iy, iz, i, j);
                    size_t x = site(L, ix, iy, iz);
                    W[(size_t)o * V + x] = (int32_t)lround(sum / (2.0 * M_PI));
                    if (near) {
                        int n = (M_PI - fabs(c1) < cut_tol) || (M_PI - fabs(c2) < cut_tol) ||
                                (M_PI - fabs(c3) < cut_tol) || (M_PI - fabs(c4) < cut_tol);
                        near[(size_t)o * V + x] = (uint8_t)n;
                    }
                }
    }
}

/* O-9  pierced-cell array.  PAPER.md:234 ("content of each cell set by the total magnitude of
 * the windings that pierce it"), :252 (one string -> value 2).  Cell x = cube [x, x+1]^3; its six
 * faces are W_xy(x), W_xy(x+z), W_yz(x), W_yz(x+x), W_zx(x), W_zx(x+y). */
void orc_cells(const orc_lattice *L, const int32_t *W, int32_t *C)
{
    size_t V = vol(L);
    for (int iz = 0; iz < L->nz; iz++)
        for (int iy = 0; iy < L->ny; iy++)
            for (int ix = 0; ix < L->nx; ix++) {
                size_t x = site(L, ix, iy, iz);
                C[x] = abs(W[0 * V + x]) + abs(W[0 * V + site(L, ix, iy, iz + 1)]) +
                       abs(W[1 * V + x]) + abs(W[1 * V + site(L, ix + 1, iy, iz)]) +
                       abs(W[2 * V + x]) + abs(W[2 * V + site(L, ix, iy + 1, iz)]);
            }
}

/* ------------------------------------------------------------------------------------------
 * O-10 / O-11  per-site densities (all WITHOUT scale-factor weights; the caller combines):
 *   kin  = |Pi|^2 + |Psi|^2
 *   grad = sum_i |D+_i phi|^2 + |D+_i psi|^2
 *   elec = sum_i E_i^2/(2 e_p0^2) + H_i^2/(2 e_q0^2)
 *   mag  = sum_{i<j} F_ij^2/(2 e_p0^2) + G_ij^2/(2 e_q0^2),  F_ij = P_ij / dx^2
 *   pot  = V(|phi|,|psi|)  of PAPER.md:52 Eq. 4 with the a=1 couplings
 *   vint = kappa0 (|phi|^2 - sigma_p^2)(|psi|^2 - sigma_q^2)
 * Lagrangian density (Eq. 1 with Eq. 12, reading R-14):
 *   L_x = kin - grad + (elec - mag)/c - c pot ;   flat-space energy density = sum of the five.
 * ---------------------------------------------------------------------------------------- */
void orc_densities(const orc_lattice *L, const orc_couplings *K, const double *state, double *kin,
                   double *grad, double *elec, double *mag, double *pot, double *vint)
{
    size_t V = vol(L);
    const double *s = state;
    double dx = L->dx;
    for (int iz = 0; iz < L->nz; iz++)
        for (int iy = 0; iy < L->ny; iy++)
            for (int ix = 0; ix < L->nx; ix++) {
                size_t x = site(L, ix, iy, iz);
                double k = 0.0, gr = 0.0, el = 0.0, mg = 0.0;
                for (int r = 0; r < 2; r++) {
                    k += s[(PIM + r) * V + x] * s[(PIM + r) * V + x];
                    k += s[(PSM + r) * V + x] * s[(PSM + r) * V + x];
                }
                for (int i = 0; i < 3; i++) {
                    double hr, hi, dr, di;
                    hop_forward(L, s + PHI * V, s + (PHI + 1) * V, s + (THA + i) * V, ix, iy, iz, i,
                                &hr, &hi);
                    dr = (hr - s[PHI * V + x]) / dx;
                    di = (hi - s[(PHI + 1) * V + x]) / dx;
                    gr += dr * dr + di * di;
                    hop_forward(L, s + PSI * V, s + (PSI + 1) * V, s + (THB + i) * V, ix, iy, iz, i,
                                &hr, &hi);
                    dr = (hr - s[PSI * V + x]) / dx;
                    di = (hi - s[(PSI + 1) * V + x]) / dx;
                    gr += dr * dr + di * di;
                    el += s[(EA + i) * V + x] * s[(EA + i) * V + x] / (2.0 * K->e1 * K->e1);
                    el += s[(HB + i) * V + x] * s[(HB + i) * V + x] / (2.0 * K->e2 * K->e2);
                }
                for (int i = 0; i < 3; i++)
                    for (int j = i + 1; j < 3; j++) {
                        double F = plaquette(L, s + THA * V, ix, iy, iz, i, j) / (dx * dx);
                        double G = plaquette(L, s + THB * V, ix, iy, iz, i, j) / (dx * dx);
                        mg += F * F / (2.0 * K->e1 * K->e1) + G * G / (2.0 * K->e2 * K->e2);
                    }
                double a2 = s[PHI * V + x] * s[PHI * V + x] +
                            s[(PHI + 1) * V + x] * s[(PHI + 1) * V + x] - K->eta1 * K->eta1;
                double b2 = s[PSI * V + x] * s[PSI * V + x] +
                            s[(PSI + 1) * V + x] * s[(PSI + 1) * V + x] - K->eta2 * K->eta2;
                kin[x] = k;
                grad[x] = gr;
                elec[x] = el;
                mag[x] = mg;
                pot[x] = 0.25 * K->lambda1 * a2 * a2 + 0.25 * K->lambda2 * b2 * b2 -
                         K->kappa * a2 * b2;
                vint[x] = K->kappa * a2 * b2;
            }
}

/* ------------------------------------------------------------------------------------------
 * Philox4x32-10 counter-based generator (Salmon, Moraes, Dror, Shaw, SC'11), restated from its
 * published definition; pinned by the known-answer vectors in tests/golden/philox_kat.txt.
 * The CUDA path carries its own independent implementation.
 * ---------------------------------------------------------------------------------------- */
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3], k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; round++) {
        uint64_t p0 = (uint64_t)0xD2511F53u * c0, p1 = (uint64_t)0xCD9E8D57u * c2;
        uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
        uint32_t n1 = (uint32_t)p1;
        uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
        uint32_t n3 = (uint32_t)p0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

static void site_random(uint64_t seed, uint64_t lin, uint32_t r[4])
{
    /* counter = (site index lo, hi, 0, 0), key = (seed lo, hi)  -- DESIGN.md section 4 */
    uint32_t ctr[4] = {(uint32_t)lin, (uint32_t)(lin >> 32), 0u, 0u};
    uint32_t key[2] = {(uint32_t)seed, (uint32_t)(seed >> 32)};
    orc_philox4x32_10(ctr, key, r);
}

/* a11 / PAPER.md:162: |phi| = sigma_p, |psi| = sigma_q, iid uniform phases; momenta, links and
 * electric fields zero (reading R-10).  phase = 2 pi r / 2^32, r0 -> phi, r1 -> psi. */
void orc_init_random_phase(const orc_lattice *L, const orc_couplings *K, uint64_t seed,
                           double *state)
{
    size_t V = vol(L);
    memset(state, 0, 20 * V * sizeof(double));
    for (size_t x = 0; x < V; x++) {
        uint32_t r[4];
        site_random(seed, (uint64_t)x, r);
        double a = 2.0 * M_PI * ((double)r[0] / 4294967296.0);
        double b = 2.0 * M_PI * ((double)r[1] / 4294967296.0);
        state[PHI * V + x] = K->eta1 * cos(a);
        state[(PHI + 1) * V + x] = K->eta1 * sin(a);
        state[PSI * V + x] = K->eta2 * cos(b);
        state[(PSI + 1) * V + x] = K->eta2 * sin(b);
    }
}

/* BASELINE.json config 3 (reading R-18): complex white noise, N(0,1) per real component by
 * Box-Muller on the site's four Philox words (u1 = (r+1)/2^32 in (0,1], u2 = r/2^32),
 * convolved with the separable periodic Gaussian exp(-d^2/(2 w^2)), |d| <= trunc, then
 * normalised to |phi| = sigma_p, |psi| = sigma_q (zero result -> phase 0). */
void orc_init_smoothed(const orc_lattice *L, const orc_couplings *K, uint64_t seed, double width,
                       int trunc, double *state)
{
    size_t V = vol(L);
    double *a = (double *)malloc(4 * V * sizeof(double));
    double *b = (double *)malloc(4 * V * sizeof(double));
    memset(state, 0, 20 * V * sizeof(double));
    for (size_t x = 0; x < V; x++) {
        uint32_t r[4];
        site_random(seed, (uint64_t)x, r);
        for (int k = 0; k < 2; k++) {
            double u1 = ((double)r[2 * k] + 1.0) / 4294967296.0;
            double u2 = (double)r[2 * k + 1] / 4294967296.0;
            double rad = sqrt(-2.0 * log(u1));
            a[(2 * k) * V + x] = rad * cos(2.0 * M_PI * u2);
            a[(2 * k + 1) * V + x] = rad * sin(2.0 * M_PI * u2);
        }
    }
    for (int dir = 0; dir < 3; dir++) {
        for (int k = 0; k < 4; k++)
            for (int iz = 0; iz < L->nz; iz++)
                for (int iy = 0; iy < L->ny; iy++)
                    for (int ix = 0; ix < L->nx; ix++) {
                        double acc = 0.0;
                        for (int d = -trunc; d <= trunc; d++)
                            acc += exp(-(double)(d * d) / (2.0 * width * width)) *
                                   a[(size_t)k * V + shift(L, ix, iy, iz, dir, d)];
                        b[(size_t)k * V + site(L, ix, iy, iz)] = acc;
                    }
        double *t = a; a = b; b = t;
    }
    for (size_t x = 0; x < V; x++) {
        double n1 = sqrt(a[x] * a[x] + a[V + x] * a[V + x]);
        double n2 = sqrt(a[2 * V + x] * a[2 * V + x] + a[3 * V + x] * a[3 * V + x]);
        state[PHI * V + x] = n1 > 0 ? K->eta1 * a[x] / n1 : K->eta1;
        state[(PHI + 1) * V + x] = n1 > 0 ? K->eta1 * a[V + x] / n1 : 0.0;
        state[PSI * V + x] = n2 > 0 ? K->eta2 * a[2 * V + x] / n2 : K->eta2;
        state[(PSI + 1) * V + x] = n2 > 0 ? K->eta2 * a[3 * V + x] / n2 : 0.0;
    }
    free(a);
    free(b);
}

/*
 * mfc_oracle.c  --  TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, fp64 CPU statement of what the hot path computes: the right-hand side of the
 * 5-equation diffuse-interface model (Allaire, K = 0; optionally the Kapila source K div(u) of Eq. 2, two
 * fluids) with stiffened-gas EOS on a uniform or non-uniform Cartesian grid (section A5c below),
 * driven by 3-stage TVD Runge-Kutta, exactly in the paper's order:
 *   ghost fill -> cons->prim -> per-direction WENO5-JS -> HLLC (+ face velocity) -> flux difference
 *   + alpha*div(u) -> RK stage combine;  plus the CFL time step.
 * Reference: /root/reference/PAPER.md (arxiv 2305.09163); every function cites the passage it follows.
 * Where the paper is silent or garbled the reading is the one listed in DESIGN.md ("Readings", B1..B21).
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may build,
 * load or call this file.  It shares no code, header, table or constant with the CUDA path
 * (paper_2305_09163_b200/csrc/), and neither includes the other.
 *
 * No blocking, fusion or reordering beyond what the algorithm states: whole-array passes, one after the
 * other.  The only parallelism is an OpenMP "parallel for" on the outermost loop of each pass (lines are
 * independent), which changes no arithmetic.  Build: gcc -O2 -ffp-contract=off [-fopenmp] -shared -fPIC.
 *
 * Parity pins (tests/test_oracle_pins.py): every function below is pinned by something other than itself
 * (closed forms, exact Riemann solutions, polynomial exactness, invariants, numpy.pad; orc_line by differencing its
 * fluxes into orc_rhs bit for bit; the mixture sound speed by a measured acoustic wave speed).  The Davis
 * wave-speed estimate and the u_face formula are pinned only through consistency/invariants (C2, C5, C7,
 * C8), not against MFC's own unpublished choice: "parity unpinned" w.r.t. MFC itself for those two readings.
 *
 * Layout: q[eq][k][j][i], i (x) fastest, padded by ng = 3 ghost cells on both sides of every active
 * dimension (PAPER.md:238 flattened arrays; PAPER.md:168 buffers).  Equation order:
 *   alpha_i rho_i (i = 1..nf), rho u_d (d = 1..ndim), rho E, alpha_i (i = 1..nf-1).      (reading B1)
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>

#define ORC_NG 3
#define ORC_MAXF 4
#define ORC_MAXEQ (2 * ORC_MAXF + 3)

typedef struct {
    int ndim;              /* 1, 2, 3 */
    int nf;                /* number of fluids */
    int n[3];              /* interior cells (1 in inactive dimensions) */
    double dx[3];          /* uniform spacing, Eq. (8) */
    double gamma[ORC_MAXF];
    double pi_inf[ORC_MAXF];
    int bc_lo[3], bc_hi[3]; /* 0 periodic, 1 extrapolation */
    double weno_eps;
    int weno_order;        /* 5 (WENO5-JS), 3 (WENO3-JS) or 1 (piecewise constant) */
    int kapila;            /* 0: Allaire model (K = 0); 1: Kapila source K div(u) on the alpha row, two fluids (Eq. 2) */
    const double *xe[3];   /* non-uniform Cartesian spacing: xe[d] = the n[d] + 2 ng + 1 cell EDGES of the padded
                              line of direction d (ghost cells included), increasing; NULL = uniform spacing dx[d] */
} orc_problem;

static int neq_of(const orc_problem *P) { return 2 * P->nf + P->ndim; }
static int pad_of(const orc_problem *P, int d) { return d < P->ndim ? P->n[d] + 2 * ORC_NG : 1; }
static size_t cells_padded(const orc_problem *P) {
    return (size_t)pad_of(P, 0) * (size_t)pad_of(P, 1) * (size_t)pad_of(P, 2);
}
/* i, j, k are padded indices */
static size_t at(const orc_problem *P, int i, int j, int k) {
    return ((size_t)k * (size_t)pad_of(P, 1) + (size_t)j) * (size_t)pad_of(P, 0) + (size_t)i;
}

int orc_neq(const orc_problem *P) { return neq_of(P); }
long long orc_elems(const orc_problem *P) { return (long long)neq_of(P) * (long long)cells_padded(P); }

/* ------------------------------------------------------------------------------------------------
 * A3. Ghost fill.  PAPER.md:168 ("allocating buffers at the domain edges", size from the WENO order).
 * Periodic: q[-m] = q[n-m], q[n-1+m] = q[m-1]; extrapolation: q[-m] = q[0], q[n-1+m] = q[n-1], m = 1..3.
 * Dimensions in order x, y, z, each pass covering the full padded extent of the other dimensions.
 * ---------------------------------------------------------------------------------------------- */
void orc_fill_ghosts(const orc_problem *P, double *q)
{
    const int neq = neq_of(P);
    const size_t C = cells_padded(P);
    for (int d = 0; d < P->ndim; ++d) {
        const int n = P->n[d];
        int ext[3] = { pad_of(P, 0), pad_of(P, 1), pad_of(P, 2) };
        ext[d] = 1;
        for (int e = 0; e < neq; ++e) {
            double *v = q + (size_t)e * C;
            for (int c = 0; c < ext[2]; ++c)
                for (int b = 0; b < ext[1]; ++b)
                    for (int a = 0; a < ext[0]; ++a)
                        for (int m = 1; m <= ORC_NG; ++m) {
                            int idx[3] = { a, b, c };
                            int src_lo = (P->bc_lo[d] == 0) ? (n - m) : 0;         /* interior index */
                            int src_hi = (P->bc_hi[d] == 0) ? (m - 1) : (n - 1);
                            size_t dst, src;
                            idx[d] = ORC_NG - m;            dst = at(P, idx[0], idx[1], idx[2]);
                            idx[d] = ORC_NG + src_lo;       src = at(P, idx[0], idx[1], idx[2]);
                            v[dst] = v[src];
                            idx[d] = ORC_NG + n - 1 + m;    dst = at(P, idx[0], idx[1], idx[2]);
                            idx[d] = ORC_NG + src_hi;       src = at(P, idx[0], idx[1], idx[2]);
                            v[dst] = v[src];
                        }
        }
    }
}

/* ------------------------------------------------------------------------------------------------
 * A2. Mixture rules for the stiffened gas, PAPER.md:54-58 (Eq. 1): rho e = p/(gamma-1) + gamma pi/(gamma-1)
 * per fluid; alpha-weighted for the mixture (reading B2): Gamma = sum alpha_i/(gamma_i-1),
 * Pi = sum alpha_i gamma_i pi_i/(gamma_i-1), alpha_nf = 1 - sum_{i<nf} alpha_i.
 * w is a primitive vector (alpha_i rho_i, u_d, p, alpha_i).
 * ---------------------------------------------------------------------------------------------- */
static void mixture(const orc_problem *P, const double *alpha_adv, double *Gam, double *Pi)
{
    const int nf = P->nf;
    double last = 1.0, G = 0.0, Q = 0.0;
    for (int i = 0; i < nf; ++i) {
        double a;
        if (i < nf - 1) { a = alpha_adv[i]; last -= a; } else { a = last; }
        G += a / (P->gamma[i] - 1.0);
        Q += a * P->gamma[i] * P->pi_inf[i] / (P->gamma[i] - 1.0);
    }
    *Gam = G; *Pi = Q;
}

/* A4. cons -> prim for one cell ("conservative variables q are converted to the primitive
 * ones before reconstruction").  w = (alpha_i rho_i, u_d = rho u_d / rho, p, alpha_i),
 * p = (rho E - rho|u|^2/2 - Pi)/Gamma. */
void orc_cons_to_prim_cell(const orc_problem *P, const double *qc, double *w)
{
    const int nf = P->nf, D = P->ndim;
    double rho = 0.0, ke = 0.0, Gam, Pi;
    for (int i = 0; i < nf; ++i) { w[i] = qc[i]; rho += qc[i]; }
    for (int d = 0; d < D; ++d) { w[nf + d] = qc[nf + d] / rho; ke += 0.5 * rho * w[nf + d] * w[nf + d]; }
    for (int i = 0; i < nf - 1; ++i) w[nf + D + 1 + i] = qc[nf + D + 1 + i];
    mixture(P, qc + nf + D + 1, &Gam, &Pi);
    w[nf + D] = (qc[nf + D] - ke - Pi) / Gam;
}

/* whole padded array */
void orc_cons_to_prim(const orc_problem *P, const double *q, double *w)
{
    const int neq = neq_of(P);
    const size_t C = cells_padded(P);
#pragma omp parallel for schedule(static)
    for (long long c = 0; c < (long long)C; ++c) {
        double qc[ORC_MAXEQ], wc[ORC_MAXEQ];
        for (int e = 0; e < neq; ++e) qc[e] = q[(size_t)e * C + (size_t)c];
        orc_cons_to_prim_cell(P, qc, wc);
        for (int e = 0; e < neq; ++e) w[(size_t)e * C + (size_t)c] = wc[e];
    }
}

/* ------------------------------------------------------------------------------------------------
 * A5. WENO5-JS, PAPER.md:143-150 (Eq. 12 with r = 0..k-1, k = 3; reading B6) and Listing 1
 * (alpha = d/(beta**2), omega = alpha/sum(alpha), v = sum(omega*poly); eps added to
 * beta, reading B8/B9).  Uniform-grid Jiang-Shu form.  Stencil a..e = w_{i-2..i+2}.
 * vL = value at face i+1/2 seen from cell i; vR = value at face i-1/2 seen from cell i.
 * ---------------------------------------------------------------------------------------------- */
void orc_weno5(double a, double b, double c, double d, double e, double eps, double *vL, double *vR)
{
    const double b0 = 13.0 / 12.0 * (a - 2.0 * b + c) * (a - 2.0 * b + c) + 0.25 * (a - 4.0 * b + 3.0 * c) * (a - 4.0 * b + 3.0 * c);
    const double b1 = 13.0 / 12.0 * (b - 2.0 * c + d) * (b - 2.0 * c + d) + 0.25 * (b - d) * (b - d);
    const double b2 = 13.0 / 12.0 * (c - 2.0 * d + e) * (c - 2.0 * d + e) + 0.25 * (3.0 * c - 4.0 * d + e) * (3.0 * c - 4.0 * d + e);
    const double d0 = 0.1, d1 = 0.6, d2 = 0.3;
    {   /* left state at i+1/2 */
        const double p0 = (2.0 * a - 7.0 * b + 11.0 * c) / 6.0;
        const double p1 = (-b + 5.0 * c + 2.0 * d) / 6.0;
        const double p2 = (2.0 * c + 5.0 * d - e) / 6.0;
        const double a0 = d0 / ((b0 + eps) * (b0 + eps));
        const double a1 = d1 / ((b1 + eps) * (b1 + eps));
        const double a2 = d2 / ((b2 + eps) * (b2 + eps));
        const double s = a0 + a1 + a2;
        *vL = (a0 / s) * p0 + (a1 / s) * p1 + (a2 / s) * p2;
    }
    {   /* right state at i-1/2: mirror image (a<->e, b<->d), so beta_2, beta_1, beta_0 pair with d0, d1, d2 */
        const double p0 = (2.0 * e - 7.0 * d + 11.0 * c) / 6.0;
        const double p1 = (-d + 5.0 * c + 2.0 * b) / 6.0;
        const double p2 = (2.0 * c + 5.0 * b - a) / 6.0;
        const double a0 = d0 / ((b2 + eps) * (b2 + eps));
        const double a1 = d1 / ((b1 + eps) * (b1 + eps));
        const double a2 = d2 / ((b0 + eps) * (b0 + eps));
        const double s = a0 + a1 + a2;
        *vR = (a0 / s) * p0 + (a1 / s) * p1 + (a2 / s) * p2;
    }
}

/* ------------------------------------------------------------------------------------------------
 * A5b. Lower-order variants of the same reconstruction (Eq. 12 with k = 2, "the third-order
 * variant", and k = 1).  WENO3-JS: two 2-cell candidates per side, ideal weights 1/3 (upwind-biased pair) and
 * 2/3 (centred pair), beta_0 = (w_i - w_{i-1})^2, beta_1 = (w_{i+1} - w_i)^2, same alpha = d / (beta + eps)^2.
 * ---------------------------------------------------------------------------------------------- */
void orc_weno3(double b, double c, double d, double eps, double *vL, double *vR)
{
    const double b0 = (c - b) * (c - b), b1 = (d - c) * (d - c);
    {   /* left state at i+1/2 */
        const double p0 = -0.5 * b + 1.5 * c, p1 = 0.5 * c + 0.5 * d;
        const double a0 = (1.0 / 3.0) / ((b0 + eps) * (b0 + eps));
        const double a1 = (2.0 / 3.0) / ((b1 + eps) * (b1 + eps));
        const double s = a0 + a1;
        *vL = (a0 / s) * p0 + (a1 / s) * p1;
    }
    {   /* right state at i-1/2: mirror image (b <-> d) */
        const double p0 = -0.5 * d + 1.5 * c, p1 = 0.5 * c + 0.5 * b;
        const double a0 = (1.0 / 3.0) / ((b1 + eps) * (b1 + eps));
        const double a1 = (2.0 / 3.0) / ((b0 + eps) * (b0 + eps));
        const double s = a0 + a1;
        *vR = (a0 / s) * p0 + (a1 / s) * p1;
    }
}

/* the reconstruction of the order the problem asks for, on the stencil a..e = w_{i-2..i+2} */
void orc_reconstruct(const orc_problem *P, double a, double b, double c, double d, double e, double *vL, double *vR)
{
    if (P->weno_order == 3) orc_weno3(b, c, d, P->weno_eps, vL, vR);
    else if (P->weno_order == 1) { *vL = c; *vR = c; }
    else orc_weno5(a, b, c, d, e, P->weno_eps, vL, vR);
}

/* ------------------------------------------------------------------------------------------------
 * A5c. WENO5-JS on a NON-UNIFORM grid ("structured mesh with non-uniform spacing"; Listing 1,
 * PAPER.md:186-220, whose per-index tables poly_coef / beta_coef / d_cb are what the formulas below evaluate to;
 * refs. [17] Jiang-Shu, [38] Shu for the general-stencil definitions; reading B20).  Written from the
 * DEFINITIONS, cell by cell, with no tables:
 *   - candidate r (r = 0, 1, 2: cells i-2..i, i-1..i+1, i..i+2) is the quadratic p_r whose cell averages over its three
 *     cells are the data: p_r = V_r' with V_r the cubic Lagrange interpolant of the primitive function
 *     V(x_{j+1/2}) = sum_{l <= j} v_l dx_l at the four edges of the stencil;
 *   - beta_r = sum_{l=1,2} dx_i^(2l-1) int_{cell i} (d^l p_r / dx^l)^2 dx  (Jiang-Shu), which for the quadratic
 *     p_r = a0 + a1 (x - x_i) + a2 (x - x_i)^2 is  a1^2 dx_i^2 + 13/3 a2^2 dx_i^4;
 *   - the ideal weights at a face are the d_r with sum_r d_r p_r(face) = p5(face), p5 the quartic with the five cell
 *     averages (V5' of the quintic interpolant at six edges): matching the coefficient of the outermost cells gives d_0 and
 *     d_2, and d_1 = 1 - d_0 - d_2;
 *   - alpha_r = d_r / (beta_r + eps)^2, omega_r = alpha_r / sum alpha, v = sum omega_r p_r(face)   (Eq. 12, Listing 1).
 * On a uniform grid this is orc_weno5 (pinned to round-off).  xe: the six edges of cells i-2..i+2; v: the five cell values.
 * ---------------------------------------------------------------------------------------------- */
/* derivative at x of the Lagrange basis polynomial m over the nodes e[0..nn-1] */
static double lagrange_d1(const double *e, int nn, int m, double x)
{
    double den = 1.0, sum = 0.0;
    for (int l = 0; l < nn; ++l) if (l != m) den *= (e[m] - e[l]);
    for (int l = 0; l < nn; ++l) {
        if (l == m) continue;
        double prod = 1.0;
        for (int q = 0; q < nn; ++q) if (q != m && q != l) prod *= (x - e[q]);
        sum += prod;
    }
    return sum / den;
}
/* second derivative at x of the CUBIC Lagrange basis polynomial m (four nodes) */
static double lagrange4_d2(const double *e, int m, double x)
{
    double den = 1.0, sum = 0.0;
    for (int l = 0; l < 4; ++l) if (l != m) { den *= (e[m] - e[l]); sum += (x - e[l]); }
    return 2.0 * sum / den;
}
/* third derivative (a constant) of the cubic Lagrange basis polynomial m */
static double lagrange4_d3(const double *e, int m)
{
    double den = 1.0;
    for (int l = 0; l < 4; ++l) if (l != m) den *= (e[m] - e[l]);
    return 6.0 / den;
}
/* value at x of the reconstruction polynomial (derivative of the interpolated primitive function) over the nc cells with
 * edges e[0..nc], written as coefficients of the cell values: p(x) = sum_j coef[j] v_j,  coef[j] = dx_j sum_{m > j} l_m'(x) */
static void recon_coef(const double *e, int nc, double x, double *coef)
{
    for (int j = 0; j < nc; ++j) {
        double s = 0.0;
        for (int m = j + 1; m <= nc; ++m) s += lagrange_d1(e, nc + 1, m, x);
        coef[j] = (e[j + 1] - e[j]) * s;
    }
}

void orc_weno5_nonuniform(const double *xe, const double *v, double eps, double *vL, double *vR)
{
    const double xm = xe[2], xp = xe[3];               /* faces i-1/2 and i+1/2 of the centre cell */
    const double dxi = xp - xm, xc = 0.5 * (xm + xp);
    double pL[3], pR[3], beta[3], c5L[5], c5R[5], dL[3], dR[3], cL[3][3], cR[3][3];
    recon_coef(xe, 5, xp, c5L);
    recon_coef(xe, 5, xm, c5R);
    for (int r = 0; r < 3; ++r) {
        const double *e = xe + r;                      /* four edges of cells i-2+r .. i+r */
        const double *w = v + r;
        recon_coef(e, 3, xp, cL[r]);
        recon_coef(e, 3, xm, cR[r]);
        pL[r] = cL[r][0] * w[0] + cL[r][1] * w[1] + cL[r][2] * w[2];
        pR[r] = cR[r][0] * w[0] + cR[r][1] * w[1] + cR[r][2] * w[2];
        /* primitive function at the four edges, V_0 = 0 */
        double V[4] = { 0.0, 0.0, 0.0, 0.0 };
        for (int m = 1; m < 4; ++m) V[m] = V[m - 1] + w[m - 1] * (e[m] - e[m - 1]);
        double a1 = 0.0, a2 = 0.0;                     /* p_r = a0 + a1 (x - xc) + a2 (x - xc)^2 */
        for (int m = 0; m < 4; ++m) {
            a1 += V[m] * lagrange4_d2(e, m, xc);
            a2 += 0.5 * V[m] * lagrange4_d3(e, m);
        }
        beta[r] = a1 * a1 * dxi * dxi + 13.0 / 3.0 * a2 * a2 * dxi * dxi * dxi * dxi;
    }
    /* ideal weights: stencil 0 alone reaches cell i-2, stencil 2 alone reaches cell i+2 */
    dL[0] = c5L[0] / cL[0][0]; dL[2] = c5L[4] / cL[2][2]; dL[1] = 1.0 - dL[0] - dL[2];
    dR[0] = c5R[0] / cR[0][0]; dR[2] = c5R[4] / cR[2][2]; dR[1] = 1.0 - dR[0] - dR[2];
    {
        double a[3], s = 0.0;
        for (int r = 0; r < 3; ++r) { a[r] = dL[r] / ((beta[r] + eps) * (beta[r] + eps)); s += a[r]; }
        *vL = (a[0] / s) * pL[0] + (a[1] / s) * pL[1] + (a[2] / s) * pL[2];
    }
    {
        double a[3], s = 0.0;
        for (int r = 0; r < 3; ++r) { a[r] = dR[r] / ((beta[r] + eps) * (beta[r] + eps)); s += a[r]; }
        *vR = (a[0] / s) * pR[0] + (a[1] / s) * pR[1] + (a[2] / s) * pR[2];
    }
}

/* the reconstruction of cell j (padded index) of a line of direction dir: uniform or non-uniform */
static void reconstruct_at(const orc_problem *P, int dir, int jpad, const double *st, double *vL, double *vR)
{
    if (P->xe[dir] && P->weno_order == 5) orc_weno5_nonuniform(P->xe[dir] + jpad - 2, st, P->weno_eps, vL, vR);
    else orc_reconstruct(P, st[0], st[1], st[2], st[3], st[4], vL, vR);
}
/* width of cell j (padded index) in direction dir */
static double cell_width(const orc_problem *P, int dir, int jpad)
{
    return P->xe[dir] ? P->xe[dir][jpad + 1] - P->xe[dir][jpad] : P->dx[dir];
}

/* ------------------------------------------------------------------------------------------------
 * A6. HLLC, PAPER.md:152-164 (Eq. 13-14), with the face velocity of PAPER.md:126-136 (Eq. 10 and the
 * garbled equation after section 3.2: the Riemann solver returns F and u; reading B5).
 *   s_L = min(u_L - c_L, u_R - c_R), s_R = max(u_L + c_L, u_R + c_R)                  (reading B11)
 *   s_* from continuity of normal velocity and pressure across the contact
 *   Eq. 14: F = F(q_K) + s_K (q*_K - q_K) in the star regions, F(q_K) when supersonic; the missing fourth
 *   case s_R <= 0 is F(q_R) (reading B7).  K = L if s_* >= 0 else R (reading B13).
 *   alpha rows carry the quasi-conservative flux alpha*u; u_face is the HLLC flux of the constant 1
 *   (reading B12), so F_alpha = alpha_K * u_face.
 * dir: 0, 1, 2 = normal direction.  wL, wR: primitive vectors.  F: neq fluxes.
 * ---------------------------------------------------------------------------------------------- */
void orc_hllc(const orc_problem *P, int dir, const double *wL, const double *wR, double *F, double *uface)
{
    const int nf = P->nf, D = P->ndim, neq = neq_of(P);
    const int iE = nf + D, iA = nf + D + 1;
    double rho[2], E[2], c[2], un[2], p[2];
    const double *w[2] = { wL, wR };
    for (int K = 0; K < 2; ++K) {
        double Gam, Pi, r = 0.0, ke = 0.0;
        for (int i = 0; i < nf; ++i) r += w[K][i];
        for (int d = 0; d < D; ++d) ke += 0.5 * r * w[K][nf + d] * w[K][nf + d];
        mixture(P, w[K] + iA, &Gam, &Pi);
        rho[K] = r;
        p[K] = w[K][iE];
        un[K] = w[K][nf + dir];
        E[K] = Gam * p[K] + Pi + ke;                                  /* A2: rho E */
        c[K] = sqrt(((Gam + 1.0) * p[K] + Pi) / (Gam * r));           /* A2: frozen mixture sound speed */
    }
    const double sL = fmin(un[0] - c[0], un[1] - c[1]);
    const double sR = fmax(un[0] + c[0], un[1] + c[1]);
    const double sS = (p[1] - p[0] + rho[0] * un[0] * (sL - un[0]) - rho[1] * un[1] * (sR - un[1]))
                    / (rho[0] * (sL - un[0]) - rho[1] * (sR - un[1]));
    const int K = (sS >= 0.0) ? 0 : 1;
    const double sK = (K == 0) ? sL : sR;
    const double shat = (K == 0) ? fmin(sL, 0.0) : fmax(sR, 0.0);
    const double xi = (sK - un[K]) / (sK - sS);
    const double *wk = w[K];
    double qK[ORC_MAXEQ], qS[ORC_MAXEQ], FK[ORC_MAXEQ];
    /* state q_K, physical flux F(q_K), star state q*_K */
    for (int i = 0; i < nf; ++i) {
        qK[i] = wk[i];
        FK[i] = wk[i] * un[K];
        qS[i] = xi * wk[i];
    }
    for (int d = 0; d < D; ++d) {
        qK[nf + d] = rho[K] * wk[nf + d];
        FK[nf + d] = rho[K] * wk[nf + d] * un[K] + ((d == dir) ? p[K] : 0.0);
        qS[nf + d] = xi * rho[K] * ((d == dir) ? sS : wk[nf + d]);
    }
    qK[iE] = E[K];
    FK[iE] = (E[K] + p[K]) * un[K];
    qS[iE] = xi * (E[K] + (sS - un[K]) * (rho[K] * sS + p[K] / (sK - un[K])));
    for (int i = 0; i < nf - 1; ++i) {
        qK[iA + i] = wk[iA + i];
        FK[iA + i] = wk[iA + i] * un[K];
        qS[iA + i] = xi * wk[iA + i];
    }
    for (int e = 0; e < neq; ++e) F[e] = FK[e] + shat * (qS[e] - qK[e]);
    *uface = un[K] + shat * (xi - 1.0);
}

/* ------------------------------------------------------------------------------------------------
 * A6b. Kapila coefficient, PAPER.md:60-62 (Eq. 2), two fluids:
 *   K = (rho_2 c_2^2 - rho_1 c_1^2) / (rho_2 c_2^2 / alpha_2 + rho_1 c_1^2 / alpha_1)
 * (the denominator of Eq. 2 prints "rho_1 c_2^2": read as rho_1 c_1^2, reading B3).  For a stiffened
 * gas (Eq. 1) c_i^2 = gamma_i (p + pi_inf_i) / rho_i, so rho_i c_i^2 = gamma_i (p + pi_inf_i).
 * ---------------------------------------------------------------------------------------------- */
double orc_kapila_K(const orc_problem *P, double alpha1, double p)
{
    const double alpha2 = 1.0 - alpha1;
    const double rc1 = P->gamma[0] * (p + P->pi_inf[0]);
    const double rc2 = P->gamma[1] * (p + P->pi_inf[1]);
    return (rc2 - rc1) / (rc2 / alpha2 + rc1 / alpha1);
}

/* ------------------------------------------------------------------------------------------------
 * A7. RHS, PAPER.md:105-130 (Eq. 6-10) with s(q) = 0 and h = -alpha on the alpha rows:
 *   L_k = sum_d (F^d_{k,-1/2} - F^d_{k,+1/2})/dx_d  [+ (alpha_i + K) * sum_d (u^d_{+1/2} - u^d_{-1/2})/dx_d]
 * K = 0 (Allaire) unless P->kapila: then the cell-centred K of Eq. 2 multiplies the same
 * face-velocity differences ("K div u").
 * Fills the ghosts of q, converts to primitives, then direction by direction: WENO on every line,
 * HLLC on every face, flux differences.  L has q's padded layout; only its interior is written.
 * ---------------------------------------------------------------------------------------------- */
void orc_rhs(const orc_problem *P, double *q, double *L)
{
    const int nf = P->nf, D = P->ndim, neq = neq_of(P);
    const size_t C = cells_padded(P);
    const int iA = nf + D + 1;
    double *w = (double *)malloc(sizeof(double) * (size_t)neq * C);
    orc_fill_ghosts(P, q);
    orc_cons_to_prim(P, q, w);
    memset(L, 0, sizeof(double) * (size_t)neq * C);

    for (int dir = 0; dir < D; ++dir) {
        const int n = P->n[dir];
        /* the two other directions, interior only */
        const int o1 = (dir + 1) % 3, o2 = (dir + 2) % 3;
        const int n1 = P->n[o1], n2 = P->n[o2];
        const int off1 = (o1 < D) ? ORC_NG : 0, off2 = (o2 < D) ? ORC_NG : 0;
#pragma omp parallel for schedule(static)
        for (int line = 0; line < n1 * n2; ++line) {
            const int b = line % n1, cidx = line / n1;
            /* per-line work arrays indexed by cell j = -1..n  ->  j+1 */
            double *vL = (double *)malloc(sizeof(double) * (size_t)(n + 2) * neq);
            double *vR = (double *)malloc(sizeof(double) * (size_t)(n + 2) * neq);
            double *Ff = (double *)malloc(sizeof(double) * (size_t)(n + 1) * neq);
            double *uf = (double *)malloc(sizeof(double) * (size_t)(n + 1));
            int idx[3];
            idx[o1] = off1 + b; idx[o2] = off2 + cidx;
            /* WENO: cells j = -1..n */
            for (int j = -1; j <= n; ++j) {
                double st[5];
                for (int e = 0; e < neq; ++e) {
                    for (int s = -2; s <= 2; ++s) {
                        idx[dir] = ORC_NG + j + s;
                        st[s + 2] = w[(size_t)e * C + at(P, idx[0], idx[1], idx[2])];
                    }
                    reconstruct_at(P, dir, ORC_NG + j, st, &vL[(size_t)(j + 1) * neq + e], &vR[(size_t)(j + 1) * neq + e]);
                }
            }
            /* HLLC: faces f = j+1/2, j = -1..n-1; left state from cell j, right state from cell j+1
             * */
            for (int j = -1; j <= n - 1; ++j)
                orc_hllc(P, dir, &vL[(size_t)(j + 1) * neq], &vR[(size_t)(j + 2) * neq],
                         &Ff[(size_t)(j + 1) * neq], &uf[j + 1]);
            /* flux difference, Eq. 9-10 */
            for (int j = 0; j < n; ++j) {
                size_t cell;
                idx[dir] = ORC_NG + j;
                cell = at(P, idx[0], idx[1], idx[2]);
                const double dxj = cell_width(P, dir, ORC_NG + j);            /* Eq. 8-9: the cell's own width */
                for (int e = 0; e < neq; ++e)
                    L[(size_t)e * C + cell] += (Ff[(size_t)j * neq + e] - Ff[(size_t)(j + 1) * neq + e]) / dxj;
                for (int i = 0; i < nf - 1; ++i) {
                    double h = q[(size_t)(iA + i) * C + cell];
                    if (P->kapila && nf == 2) h += orc_kapila_K(P, w[(size_t)iA * C + cell], w[(size_t)(nf + D) * C + cell]);
                    L[(size_t)(iA + i) * C + cell] += h * (uf[j + 1] - uf[j]) / dxj;
                }
            }
            free(vL); free(vR); free(Ff); free(uf);
        }
    }
    free(w);
}

/* one direction's reconstructed states and fluxes on a single 1-D line of primitives, for unit pins and
 * stage-by-stage parity: w[neq][n + 2 ng] -> vL, vR [neq][n+2] (cells -1..n), F [neq][n+1], uf [n+1] */
void orc_line(const orc_problem *P, int dir, int n, const double *w, double *vL, double *vR, double *F, double *uf)
{
    const int neq = neq_of(P);
    const int np = n + 2 * ORC_NG;
    for (int j = -1; j <= n; ++j)
        for (int e = 0; e < neq; ++e) {
            const double *s = w + (size_t)e * np + ORC_NG + j;
            reconstruct_at(P, dir, ORC_NG + j, s - 2, &vL[(size_t)e * (n + 2) + j + 1], &vR[(size_t)e * (n + 2) + j + 1]);
        }
    for (int j = -1; j <= n - 1; ++j) {
        double wl[ORC_MAXEQ], wr[ORC_MAXEQ], f[ORC_MAXEQ];
        for (int e = 0; e < neq; ++e) { wl[e] = vL[(size_t)e * (n + 2) + j + 1]; wr[e] = vR[(size_t)e * (n + 2) + j + 2]; }
        orc_hllc(P, dir, wl, wr, f, &uf[j + 1]);
        for (int e = 0; e < neq; ++e) F[(size_t)e * (n + 1) + j + 1] = f[e];
    }
}

/* ------------------------------------------------------------------------------------------------
 * A8. 3-stage TVD (SSP) Runge-Kutta, PAPER.md:172 (ref. [19]; reading B16):
 *   q1 = q + dt L(q);  q2 = 3/4 q + 1/4 (q1 + dt L(q1));  q <- 1/3 q + 2/3 (q2 + dt L(q2)).
 * Interior cells only are updated; ghosts are refilled inside every L.
 * ---------------------------------------------------------------------------------------------- */
void orc_rk3_step(const orc_problem *P, double *q, double dt)
{
    const size_t N = (size_t)orc_elems(P);
    double *q1 = (double *)malloc(sizeof(double) * N);
    double *q2 = (double *)malloc(sizeof(double) * N);
    double *L = (double *)malloc(sizeof(double) * N);
    orc_rhs(P, q, L);
#pragma omp parallel for schedule(static)
    for (long long i = 0; i < (long long)N; ++i) q1[i] = q[i] + dt * L[i];
    orc_rhs(P, q1, L);
#pragma omp parallel for schedule(static)
    for (long long i = 0; i < (long long)N; ++i) q2[i] = 0.75 * q[i] + 0.25 * (q1[i] + dt * L[i]);
    orc_rhs(P, q2, L);
#pragma omp parallel for schedule(static)
    for (long long i = 0; i < (long long)N; ++i) q[i] = (1.0 / 3.0) * q[i] + (2.0 / 3.0) * (q2[i] + dt * L[i]);
    free(q1); free(q2); free(L);
}

/* ------------------------------------------------------------------------------------------------
 * A9. CFL time step ("CFL-restricted time step"; reading B17):
 *   dt = cfl * min over interior cells and directions of dx_d / (|u_d| + c), dx_d the cell's own width.
 * ---------------------------------------------------------------------------------------------- */
double orc_cfl_dt(const orc_problem *P, const double *q, double cfl)
{
    const int nf = P->nf, D = P->ndim, neq = neq_of(P);
    const size_t C = cells_padded(P);
    double best = INFINITY;
    for (int k = 0; k < P->n[2]; ++k)
        for (int j = 0; j < P->n[1]; ++j)
            for (int i = 0; i < P->n[0]; ++i) {
                double qc[ORC_MAXEQ], w[ORC_MAXEQ], Gam, Pi, rho = 0.0, c;
                size_t cell = at(P, i + ORC_NG, j + (D > 1 ? ORC_NG : 0), k + (D > 2 ? ORC_NG : 0));
                for (int e = 0; e < neq; ++e) qc[e] = q[(size_t)e * C + cell];
                orc_cons_to_prim_cell(P, qc, w);
                for (int f = 0; f < nf; ++f) rho += w[f];
                mixture(P, w + nf + D + 1, &Gam, &Pi);
                c = sqrt(((Gam + 1.0) * w[nf + D] + Pi) / (Gam * rho));
                for (int d = 0; d < D; ++d) {
                    const int jp = (d == 0 ? i : d == 1 ? j : k) + ORC_NG;
                    double t = cell_width(P, d, jp) / (fabs(w[nf + d]) + c);
                    if (t < best) best = t;
                }
            }
    return cfl * best;
}

#ifdef _OPENMP
#include <omp.h>
int orc_threads(void) { return omp_get_max_threads(); }
void orc_set_threads(int n) { omp_set_num_threads(n); }
#else
int orc_threads(void) { return 1; }
void orc_set_threads(int n) { (void)n; }
#endif

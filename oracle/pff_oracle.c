/*
 * pff_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, single-threaded fp64 CPU restatement of the explicit phase-field
 * fracture step of arxiv/paper_2606_23458 ("A matrix-free, differentiable PyTorch
 * solver for phase-field fracture"), written from /root/reference/PAPER.md.
 * It exists only so that tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference leg can check and time the CUDA library against it.
 * It shares no code, header, table or helper with paper_2606_23458_b200/csrc and is
 * never called by the product path.
 *
 * Conventions: user numbering, AoS arrays (xy[N][2], u[N][2], tri[Ne][3]), SI units,
 * unit thickness.  Loops are written in the paper's order (element gather -> element
 * math -> scatter) with no blocking, fusion or reordering.
 *
 * Citations are PAPER.md line numbers + equation.  Readings of points where the
 * paper is silent are the ones listed in DESIGN.md ("Readings", R1..R14) and
 * SURVEY.md 8(c); each is marked [Rk] below.
 *
 * Pin status (tests/test_oracle_*.py, all -m "not gpu"):
 *   geometry / strain / force        pinned: Eq. 9 reference triangle, patch test, rigid body, FD of energy
 *   spectral, vol-dev, isotropic     pinned: psi+ + psi- = psi, numpy eigh restatement, hand values, FD of energy
 *   star-convex split                psi+ + psi- = psi, gamma*=0 == vol-dev, gamma*=-1 == isotropic, FD pinned;
 *                                    fidelity to the paper's own code: PARITY UNPINNED (PAPER.md gives no formula) [R5]
 *   d_e = centroid mean in g(d)      PARITY UNPINNED vs the paper's code (paper silent) [R3]
 *   H per element                    PARITY UNPINNED vs the paper's code (paper writes H(x,t)) [R2]
 *   velocity-Verlet                  pinned: shadow-energy conservation, momentum balance, free flight
 *   damage operator / rhs / diag     pinned: textbook P1 stencils, dense assembly, 1-D AT2 cosh profile, AT1 exact profile
 *   AT1 projected PCG                pinned: brute-force active-set enumeration, projected Gauss-Seidel, KKT residuals
 *   energies                         pinned: closed forms
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

typedef struct {
    double E, nu, rho, Gc, l0, eta, gamma_star;
    int model; /* 1 = AT1, 2 = AT2                         (L69)  */
    int split; /* 0 iso, 1 spectral, 2 vol-dev, 3 star-convex (L71-79, L85) */
    int plane; /* 0 plane strain, 1 plane stress            (L85)  */
} orc_material;

static double pos(double x) { return x > 0.0 ? x : 0.0; } /* <x>_+ */
static double neg(double x) { return x < 0.0 ? x : 0.0; } /* <x>_- */

/* ---- material constants, L85 ------------------------------------------------ */
static double lame_mu(const orc_material *m) { return m->E / (2.0 * (1.0 + m->nu)); }
static double lame_lambda(const orc_material *m)
{
    if (m->plane == 1) return m->E * m->nu / (1.0 - m->nu * m->nu);          /* lambda_PS */
    return m->E * m->nu / ((1.0 + m->nu) * (1.0 - 2.0 * m->nu));             /* lambda_PE */
}
static double bulk_K(const orc_material *m) { return m->E / (3.0 * (1.0 - 2.0 * m->nu)); }
/* eps_zz = c * tr_2D(eps):  c = 0 in plane strain, -nu/(1-nu) in plane stress (L85) */
static double ezz_factor(const orc_material *m) { return m->plane == 1 ? -m->nu / (1.0 - m->nu) : 0.0; }

/* ---- geometry, Eq. 9 (L120-124) ---------------------------------------------
 * tri_out receives the connectivity re-oriented counter-clockwise [R1]: nodes 2 and 3
 * are swapped when the signed area is negative, so that A_e > 0.
 * gradphi[e][i] = (d_x phi_i, d_y phi_i).  Returns 0, or 1+e for a degenerate element. */
int orc_geometry(int64_t n_nodes, const double *xy, int64_t n_elems, const int32_t *tri,
                 int32_t *tri_out, double *gradphi, double *area)
{
    for (int64_t e = 0; e < n_elems; ++e) {
        int32_t n1 = tri[3 * e], n2 = tri[3 * e + 1], n3 = tri[3 * e + 2];
        if (n1 < 0 || n2 < 0 || n3 < 0 || n1 >= n_nodes || n2 >= n_nodes || n3 >= n_nodes) return (int)(1 + e);
        double x1 = xy[2 * n1], y1 = xy[2 * n1 + 1];
        double x2 = xy[2 * n2], y2 = xy[2 * n2 + 1];
        double x3 = xy[2 * n3], y3 = xy[2 * n3 + 1];
        double twoA = (x2 - x1) * (y3 - y1) - (x3 - x1) * (y2 - y1);
        if (twoA < 0.0) { /* [R1] swap local nodes 2 and 3 */
            int32_t t = n2; n2 = n3; n3 = t;
            double tx = x2; x2 = x3; x3 = tx;
            double ty = y2; y2 = y3; y3 = ty;
            twoA = -twoA;
        }
        double l12 = (x2 - x1) * (x2 - x1) + (y2 - y1) * (y2 - y1);
        double l23 = (x3 - x2) * (x3 - x2) + (y3 - y2) * (y3 - y2);
        double l31 = (x1 - x3) * (x1 - x3) + (y1 - y3) * (y1 - y3);
        double lmax = fmax(l12, fmax(l23, l31));
        if (!(0.5 * twoA > 1e-14 * lmax)) return (int)(1 + e);
        tri_out[3 * e] = n1; tri_out[3 * e + 1] = n2; tri_out[3 * e + 2] = n3;
        area[e] = 0.5 * twoA;
        double *g = gradphi + 6 * e;
        g[0] = (y2 - y3) / twoA; g[1] = (x3 - x2) / twoA;
        g[2] = (y3 - y1) / twoA; g[3] = (x1 - x3) / twoA;
        g[4] = (y1 - y2) / twoA; g[5] = (x2 - x1) / twoA;
    }
    return 0;
}

/* lumped mass m_i = rho * sum_{e contains i} A_e / 3   (L169) */
void orc_lumped_mass(int64_t n_nodes, int64_t n_elems, const int32_t *tri, const double *area,
                     double rho, double *mass)
{
    for (int64_t i = 0; i < n_nodes; ++i) mass[i] = 0.0;
    for (int64_t e = 0; e < n_elems; ++e)
        for (int k = 0; k < 3; ++k) mass[tri[3 * e + k]] += rho * area[e] / 3.0;
}

/* h_min = minimum element incircle diameter = 4 A / perimeter   (L169) */
double orc_hmin(int64_t n_elems, const int32_t *tri, const double *xy, const double *area)
{
    double h = INFINITY;
    for (int64_t e = 0; e < n_elems; ++e) {
        const int32_t *t = tri + 3 * e;
        double per = 0.0;
        for (int k = 0; k < 3; ++k) {
            int32_t a = t[k], b = t[(k + 1) % 3];
            per += hypot(xy[2 * a] - xy[2 * b], xy[2 * a + 1] - xy[2 * b + 1]);
        }
        double he = 4.0 * area[e] / per;
        if (he < h) h = he;
    }
    return h;
}

/* CFL: dt_crit = h_min / c_p,  c_p = sqrt((lambda + 2 mu) / rho)  (L169); the caller applies alpha */
double orc_dt_crit(const orc_material *m, double hmin)
{
    double cp = sqrt((lame_lambda(m) + 2.0 * lame_mu(m)) / m->rho);
    return hmin / cp;
}

/* ---- element response ---------------------------------------------------------
 * In: in-plane strain (exx, eyy, exy) with exy the tensor component.
 * Out: psi+ and psi- (undegraded), and the degraded in-plane Cauchy stress
 *      sigma = g dpsi+/deps + dpsi-/deps  (L93),  g = (1 - d)^2 + eta  (L79).        */
void orc_element_response(const orc_material *m, double exx, double eyy, double exy, double g,
                          double *psi_p, double *psi_m, double sig[3])
{
    const double mu = lame_mu(m);
    if (m->split == 1) {
        /* Spectral split, Eq. 2 (L71-75).  Principal strains and directions of the 2x2
         * strain by the Mohr-circle construction; stress assembled from the spectral
         * representation  sigma+- = lambda <tr>+- I + 2 mu sum_a <eps_a>+- n_a (x) n_a. */
        const double lam = lame_lambda(m);
        double theta = 0.5 * atan2(2.0 * exy, exx - eyy);
        double c = cos(theta), s = sin(theta);
        double n[2][2] = {{c, s}, {-s, c}};
        double ev[2];
        for (int a = 0; a < 2; ++a)
            ev[a] = n[a][0] * (exx * n[a][0] + exy * n[a][1]) + n[a][1] * (exy * n[a][0] + eyy * n[a][1]);
        double tr = exx + eyy;
        *psi_p = 0.5 * lam * pos(tr) * pos(tr) + mu * (pos(ev[0]) * pos(ev[0]) + pos(ev[1]) * pos(ev[1]));
        *psi_m = 0.5 * lam * neg(tr) * neg(tr) + mu * (neg(ev[0]) * neg(ev[0]) + neg(ev[1]) * neg(ev[1]));
        double sp[3] = {lam * pos(tr), lam * pos(tr), 0.0}, sm[3] = {lam * neg(tr), lam * neg(tr), 0.0};
        for (int a = 0; a < 2; ++a) {
            double nn[3] = {n[a][0] * n[a][0], n[a][1] * n[a][1], n[a][0] * n[a][1]};
            for (int k = 0; k < 3; ++k) {
                sp[k] += 2.0 * mu * pos(ev[a]) * nn[k];
                sm[k] += 2.0 * mu * neg(ev[a]) * nn[k];
            }
        }
        for (int k = 0; k < 3; ++k) sig[k] = g * sp[k] + sm[k];
        return;
    }
    if (m->split == 0) {
        /* Isotropic: psi+ = psi, psi- = 0 (L79); psi = lambda/2 tr^2 + mu eps:eps with the
         * plane-assumption lambda (L85). */
        const double lam = lame_lambda(m);
        double tr = exx + eyy;
        *psi_p = 0.5 * lam * tr * tr + mu * (exx * exx + eyy * eyy + 2.0 * exy * exy);
        *psi_m = 0.0;
        sig[0] = g * (lam * tr + 2.0 * mu * exx);
        sig[1] = g * (lam * tr + 2.0 * mu * eyy);
        sig[2] = g * (2.0 * mu * exy);
        return;
    }
    /* Volumetric-deviatoric split, Eq. 3 (L75-79), and its star-convex variant [R5], on the
     * 3-D strain: eps_zz = c tr_2D (L85), 3-D bulk modulus K.
     *   psi+ = K/2 (<tr>+^2 - gamma* <tr>-^2) + mu e:e,   psi- = (1 + gamma*) K/2 <tr>-^2
     * (gamma* = 0 is Amor).  The in-plane stress is the derivative with eps_zz slaved [R4]:
     *   sigma_ab = s3_ab + c s3_zz delta_ab,   s3 = dpsi/d(eps_3D).                          */
    const double K = bulk_K(m), cz = ezz_factor(m);
    const double gs = (m->split == 3) ? m->gamma_star : 0.0;
    double e3[3][3] = {{exx, exy, 0.0}, {exy, eyy, 0.0}, {0.0, 0.0, cz * (exx + eyy)}};
    double tr = e3[0][0] + e3[1][1] + e3[2][2];
    double dev[3][3], dd = 0.0;
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j) {
            dev[i][j] = e3[i][j] - (i == j ? tr / 3.0 : 0.0);
            dd += dev[i][j] * dev[i][j];
        }
    *psi_p = 0.5 * K * (pos(tr) * pos(tr) - gs * neg(tr) * neg(tr)) + mu * dd;
    *psi_m = (1.0 + gs) * 0.5 * K * neg(tr) * neg(tr);
    double phyd = g * K * (pos(tr) - gs * neg(tr)) + (1.0 + gs) * K * neg(tr);
    double s3[3][3];
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j) s3[i][j] = (i == j ? phyd : 0.0) + 2.0 * mu * g * dev[i][j];
    sig[0] = s3[0][0] + cz * s3[2][2];
    sig[1] = s3[1][1] + cz * s3[2][2];
    sig[2] = s3[0][1];
}

/* element strain from nodal displacements: eps = sym(grad u), constant per P1 element (L69, L42) */
static void element_strain(const int32_t *t, const double *g, const double *u, double *exx, double *eyy, double *exy)
{
    double a = 0.0, b = 0.0, c = 0.0;
    for (int i = 0; i < 3; ++i) {
        double ux = u[2 * t[i]], uy = u[2 * t[i] + 1];
        a += g[2 * i] * ux;
        b += g[2 * i + 1] * uy;
        c += 0.5 * (g[2 * i + 1] * ux + g[2 * i] * uy);
    }
    *exx = a; *eyy = b; *exy = c;
}

/* degradation at the element: g = (1 - d_e)^2 + eta with d_e the centroid value [R3] (L79) */
static double element_g(const orc_material *m, const int32_t *t, const double *d)
{
    double de = (d[t[0]] + d[t[1]] + d[t[2]]) / 3.0;
    return (1.0 - de) * (1.0 - de) + m->eta;
}

/* internal force f_int(u, d) (L42-43, L124): f_i^e = A_e sigma . grad phi_i, scattered to nodes.
 * psi_plus[e] (may be NULL) receives the undegraded tensile energy density.               */
void orc_internal_force(int64_t n_nodes, int64_t n_elems, const int32_t *tri, const double *gradphi,
                        const double *area, const orc_material *m, const double *u, const double *d,
                        double *f, double *psi_plus)
{
    for (int64_t i = 0; i < 2 * n_nodes; ++i) f[i] = 0.0;
    for (int64_t e = 0; e < n_elems; ++e) {
        const int32_t *t = tri + 3 * e;
        const double *g = gradphi + 6 * e;
        double exx, eyy, exy, pp, pm, s[3];
        element_strain(t, g, u, &exx, &eyy, &exy);
        orc_element_response(m, exx, eyy, exy, element_g(m, t, d), &pp, &pm, s);
        for (int i = 0; i < 3; ++i) {
            f[2 * t[i]]     += area[e] * (s[0] * g[2 * i] + s[2] * g[2 * i + 1]);
            f[2 * t[i] + 1] += area[e] * (s[2] * g[2 * i] + s[1] * g[2 * i + 1]);
        }
        if (psi_plus) psi_plus[e] = pp;
    }
}

/* consistent nodal load of a traction t on boundary edges: each end node gets t L / 2 [R8] (Eq. 5) */
void orc_traction(int64_t n_edges, const int32_t *edge_nodes, const double *t, const double *xy, double *fext)
{
    for (int64_t k = 0; k < n_edges; ++k) {
        int32_t a = edge_nodes[2 * k], b = edge_nodes[2 * k + 1];
        double L = hypot(xy[2 * a] - xy[2 * b], xy[2 * a + 1] - xy[2 * b + 1]);
        for (int c = 0; c < 2; ++c) {
            fext[2 * a + c] += 0.5 * L * t[2 * k + c];
            fext[2 * b + c] += 0.5 * L * t[2 * k + c];
        }
    }
}

/* a = m^-1 (S f_ext - f_int(u, d)), zero on Dirichlet dofs [R8]; used for a_0 and inside the step */
static void acceleration(int64_t n_nodes, int64_t n_elems, const int32_t *tri, const double *gradphi,
                         const double *area, const double *mass, const orc_material *m, const double *u,
                         const double *d, const double *fext, double S, int64_t n_dir, const int32_t *dir_dof,
                         double *a_out, double *psi_plus, double *fwork)
{
    orc_internal_force(n_nodes, n_elems, tri, gradphi, area, m, u, d, fwork, psi_plus);
    for (int64_t i = 0; i < n_nodes; ++i)
        for (int c = 0; c < 2; ++c) a_out[2 * i + c] = (S * fext[2 * i + c] - fwork[2 * i + c]) / mass[i];
    for (int64_t k = 0; k < n_dir; ++k) a_out[dir_dof[k]] = 0.0;
}

void orc_init_accel(int64_t n_nodes, int64_t n_elems, const int32_t *tri, const double *gradphi,
                    const double *area, const double *mass, const orc_material *m, const double *u,
                    const double *d, const double *fext, double S, int64_t n_dir, const int32_t *dir_dof, double *a)
{
    double *fw = (double *)malloc(sizeof(double) * 2 * n_nodes);
    acceleration(n_nodes, n_elems, tri, gradphi, area, mass, m, u, d, fext, S, n_dir, dir_dof, a, NULL, fw);
    free(fw);
}

/* One explicit step n -> n+1 (L114, L161-167), d fixed at d_n:
 *   Eq. 16  u <- u + dt v + dt^2/2 a ; Dirichlet dofs overwritten with u_bar(t_{n+1})   [R8]
 *   Eq. 17  a+ = m^-1 (S(t_{n+1}) f_ext - f_int(u, d_n)) ; a+ = 0 on Dirichlet dofs
 *   Eq. 18  v <- v + dt/2 (a + a+) ; v = v_bar on Dirichlet dofs ; a <- a+
 *   history H_e <- max(H_e, psi+_e)  (L98, L114), one value per element [R2]              */
void orc_explicit_step(int64_t n_nodes, int64_t n_elems, const int32_t *tri, const double *gradphi,
                       const double *area, const double *mass, const orc_material *m, double *u, double *v,
                       double *a, const double *d, double *H, const double *fext, double S, double dt,
                       int64_t n_dir, const int32_t *dir_dof, const double *dir_u, const double *dir_v)
{
    double *anew = (double *)malloc(sizeof(double) * 2 * n_nodes);
    double *fw = (double *)malloc(sizeof(double) * 2 * n_nodes);
    double *pp = (double *)malloc(sizeof(double) * n_elems);
    for (int64_t i = 0; i < 2 * n_nodes; ++i) u[i] = u[i] + dt * v[i] + 0.5 * dt * dt * a[i];
    for (int64_t k = 0; k < n_dir; ++k) u[dir_dof[k]] = dir_u[k];
    acceleration(n_nodes, n_elems, tri, gradphi, area, mass, m, u, d, fext, S, n_dir, dir_dof, anew, pp, fw);
    for (int64_t i = 0; i < 2 * n_nodes; ++i) {
        v[i] = v[i] + 0.5 * dt * (a[i] + anew[i]);
        a[i] = anew[i];
    }
    for (int64_t k = 0; k < n_dir; ++k) v[dir_dof[k]] = dir_v[k];
    for (int64_t e = 0; e < n_elems; ++e)
        if (pp[e] > H[e]) H[e] = pp[e];
    free(anew); free(fw); free(pp);
}

/* ---- damage sub-problem (L98-112, L173, L185) -----------------------------------
 * AT2 (Eq. 6): (Gc/l0 + 2H) d - Gc l0 Lap d = 2H
 * AT1 (Eq. 8): 2H d - 3/4 Gc l0 Lap d >= 2H - 3 Gc/(8 l0)
 * P1 Galerkin with the CONSISTENT element mass M^e_ij = A_e (1 + delta_ij)/12 (L185) for the
 * reaction term and K^e_ij = A_e grad phi_i . grad phi_j for the diffusion term [R9].        */
static void damage_coeffs(const orc_material *m, double He, double *c_react, double *kappa, double *src)
{
    if (m->model == 2) { *c_react = m->Gc / m->l0 + 2.0 * He; *kappa = m->Gc * m->l0; *src = 2.0 * He; }
    else { *c_react = 2.0 * He; *kappa = 0.75 * m->Gc * m->l0; *src = 2.0 * He - 3.0 * m->Gc / (8.0 * m->l0); }
}

/* q = A p, matrix-free gather - compute - scatter (L173) */
void orc_damage_matvec(int64_t n_nodes, int64_t n_elems, const int32_t *tri, const double *gradphi,
                       const double *area, const orc_material *m, const double *H, const double *p, double *q)
{
    for (int64_t i = 0; i < n_nodes; ++i) q[i] = 0.0;
    for (int64_t e = 0; e < n_elems; ++e) {
        const int32_t *t = tri + 3 * e;
        const double *g = gradphi + 6 * e;
        double c, kap, src;
        damage_coeffs(m, H[e], &c, &kap, &src);
        double pe[3] = {p[t[0]], p[t[1]], p[t[2]]};
        double gx = 0.0, gy = 0.0; /* grad p_e */
        for (int j = 0; j < 3; ++j) { gx += g[2 * j] * pe[j]; gy += g[2 * j + 1] * pe[j]; }
        for (int i = 0; i < 3; ++i) {
            double react = 0.0;
            for (int j = 0; j < 3; ++j) react += area[e] * ((i == j) ? 2.0 : 1.0) / 12.0 * pe[j];
            q[t[i]] += c * react + kap * area[e] * (g[2 * i] * gx + g[2 * i + 1] * gy);
        }
    }
}

/* right-hand side b_i = sum_e s_e A_e / 3 and Jacobi diagonal D_i = A_ii */
void orc_damage_rhs_diag(int64_t n_nodes, int64_t n_elems, const int32_t *tri, const double *gradphi,
                         const double *area, const orc_material *m, const double *H, double *b, double *D)
{
    for (int64_t i = 0; i < n_nodes; ++i) { b[i] = 0.0; D[i] = 0.0; }
    for (int64_t e = 0; e < n_elems; ++e) {
        const int32_t *t = tri + 3 * e;
        const double *g = gradphi + 6 * e;
        double c, kap, src;
        damage_coeffs(m, H[e], &c, &kap, &src);
        for (int i = 0; i < 3; ++i) {
            b[t[i]] += src * area[e] / 3.0;
            D[t[i]] += c * area[e] / 6.0 + kap * area[e] * (g[2 * i] * g[2 * i] + g[2 * i + 1] * g[2 * i + 1]);
        }
    }
}

static double dotF(int64_t n, const double *a, const double *b, const unsigned char *F)
{
    double s = 0.0;
    for (int64_t i = 0; i < n; ++i) if (F[i]) s += a[i] * b[i];
    return s;
}

/* Damage solve for d_{n+1} given H_{n+1} and d_n (in d, overwritten) [R10-R12].
 *   AT2: Jacobi-PCG from x0 = d_n on the non-Dirichlet nodes (L173, L177, L468), then
 *        d+ = min(1, max(d_n, d*))                                            (L179)
 *   AT1: projected Jacobi-PCG with lower bound lb = d_n (>= 0): nodes at the bound with
 *        negative residual are frozen, CG runs on the free set, restart when the set
 *        changes (L181); result = minimiser of 1/2 d'Ad - b'd s.t. d >= lb; then min(.,1).
 * Damage-Dirichlet nodes keep their value. Stopping [R10]: ||r_F||_2 <= rel_tol * nb with
 * nb = max(||b||_2, ||b - A x0||_2 over the non-Dirichlet nodes, 1e-300).
 * Returns 0 if converged, 5 if max_iter mat-vecs were used (result still written).           */
int orc_damage_solve(int64_t n_nodes, int64_t n_elems, const int32_t *tri, const double *gradphi,
                     const double *area, const orc_material *m, const double *H, double *d,
                     int64_t n_ddir, const int32_t *ddir_node, double rel_tol, int max_iter,
                     int *iters_out, double *relres_out)
{
    int64_t n = n_nodes;
    double *b = malloc(sizeof(double) * n), *D = malloc(sizeof(double) * n), *x = malloc(sizeof(double) * n);
    double *r = malloc(sizeof(double) * n), *z = malloc(sizeof(double) * n), *p = malloc(sizeof(double) * n);
    double *q = malloc(sizeof(double) * n), *lb = malloc(sizeof(double) * n);
    unsigned char *F = malloc(n), *fixed = calloc(n, 1);
    const int projected = (m->model == 1);
    int iters = 0, status = 5;
    double relres = 0.0;

    orc_damage_rhs_diag(n_nodes, n_elems, tri, gradphi, area, m, H, b, D);
    for (int64_t k = 0; k < n_ddir; ++k) fixed[ddir_node[k]] = 1;
    for (int64_t i = 0; i < n; ++i) { lb[i] = projected ? d[i] : -INFINITY; x[i] = d[i]; }
    double nb = 0.0;
    for (int64_t i = 0; i < n; ++i) nb += b[i] * b[i];
    nb = fmax(sqrt(nb), 1e-300);

    for (int pass = 0;; ++pass) { /* restart loop */
        orc_damage_matvec(n_nodes, n_elems, tri, gradphi, area, m, H, x, q);
        for (int64_t i = 0; i < n; ++i) r[i] = b[i] - q[i];
        if (pass == 0) {
            double n0 = 0.0;
            for (int64_t i = 0; i < n; ++i) if (!fixed[i]) n0 += r[i] * r[i];
            nb = fmax(nb, sqrt(n0));
        }
        for (int64_t i = 0; i < n; ++i) F[i] = !fixed[i] && (x[i] > lb[i] || r[i] > 0.0);
        relres = sqrt(dotF(n, r, r, F)) / nb;
        if (relres <= rel_tol) { status = 0; break; }
        if (iters >= max_iter) break;
        for (int64_t i = 0; i < n; ++i) { z[i] = F[i] ? r[i] / D[i] : 0.0; p[i] = z[i]; }
        double rho = dotF(n, r, z, F);
        int restart = 0;
        while (!restart && iters < max_iter) {
            orc_damage_matvec(n_nodes, n_elems, tri, gradphi, area, m, H, p, q);
            ++iters;
            double alpha = rho / dotF(n, p, q, F);
            double amax = INFINITY;
            for (int64_t i = 0; i < n; ++i)
                if (F[i] && p[i] < 0.0) { double s = (lb[i] - x[i]) / p[i]; if (s < amax) amax = s; }
            if (alpha >= amax) { /* step hits a bound first: truncate, snap, restart */
                for (int64_t i = 0; i < n; ++i) {
                    if (!F[i]) continue;
                    x[i] += amax * p[i];
                    if (p[i] < 0.0 && x[i] <= lb[i] + 1e-15 * fabs(lb[i])) x[i] = lb[i];
                    if (x[i] < lb[i]) x[i] = lb[i];
                }
                restart = 1;
                break;
            }
            for (int64_t i = 0; i < n; ++i) { x[i] += alpha * p[i]; r[i] -= alpha * q[i]; }
            relres = sqrt(dotF(n, r, r, F)) / nb;
            if (relres <= rel_tol) { restart = 1; break; } /* re-derive F from the true residual */
            for (int64_t i = 0; i < n; ++i) z[i] = F[i] ? r[i] / D[i] : 0.0;
            double rho1 = dotF(n, r, z, F);
            double beta = rho1 / rho;
            for (int64_t i = 0; i < n; ++i) p[i] = z[i] + beta * p[i];
            rho = rho1;
        }
        if (!restart) break; /* max_iter */
    }
    for (int64_t i = 0; i < n; ++i) {
        if (fixed[i]) continue;
        double xi = x[i];
        if (xi < d[i]) xi = d[i]; /* irreversibility d+ >= d_n (L179) */
        if (xi > 1.0) xi = 1.0;
        d[i] = xi;
    }
    if (iters_out) *iters_out = iters;
    if (relres_out) *relres_out = relres;
    free(b); free(D); free(x); free(r); free(z); free(p); free(q); free(lb); free(F); free(fixed);
    return status;
}

/* ---- energies per unit thickness (Eq. 1) ------------------------
 * out = { E_el, E_kin, E_frac, E_tot }
 *   E_el   = sum_e A_e (g(d_e) psi+ + psi-)
 *   E_kin  = 1/2 sum_i m_i |v_i|^2                       (lumped mass, L169)
 *   AT2: E_frac = Gc sum_e [ d^e' M^e d^e / (2 l0) + l0/2 A_e |grad d_e|^2 ]
 *   AT1: E_frac = 3 Gc / 8 sum_e [ A_e mean(d^e) / l0 + l0 A_e |grad d_e|^2 ]                */
void orc_energies(int64_t n_nodes, int64_t n_elems, const int32_t *tri, const double *gradphi,
                  const double *area, const double *mass, const orc_material *m, const double *u,
                  const double *v, const double *d, double out[4])
{
    double Eel = 0.0, Ekin = 0.0, Efr = 0.0;
    for (int64_t e = 0; e < n_elems; ++e) {
        const int32_t *t = tri + 3 * e;
        const double *g = gradphi + 6 * e;
        double exx, eyy, exy, pp, pm, s[3];
        element_strain(t, g, u, &exx, &eyy, &exy);
        double ge = element_g(m, t, d);
        orc_element_response(m, exx, eyy, exy, ge, &pp, &pm, s);
        Eel += area[e] * (ge * pp + pm);
        double de[3] = {d[t[0]], d[t[1]], d[t[2]]};
        double gx = 0.0, gy = 0.0;
        for (int j = 0; j < 3; ++j) { gx += g[2 * j] * de[j]; gy += g[2 * j + 1] * de[j]; }
        if (m->model == 2) {
            double dMd = 0.0;
            for (int i = 0; i < 3; ++i)
                for (int j = 0; j < 3; ++j) dMd += de[i] * area[e] * ((i == j) ? 2.0 : 1.0) / 12.0 * de[j];
            Efr += m->Gc * (dMd / (2.0 * m->l0) + 0.5 * m->l0 * area[e] * (gx * gx + gy * gy));
        } else {
            double dbar = (de[0] + de[1] + de[2]) / 3.0;
            Efr += 0.375 * m->Gc * (area[e] * dbar / m->l0 + m->l0 * area[e] * (gx * gx + gy * gy));
        }
    }
    for (int64_t i = 0; i < n_nodes; ++i)
        Ekin += 0.5 * mass[i] * (v[2 * i] * v[2 * i] + v[2 * i + 1] * v[2 * i + 1]);
    out[0] = Eel; out[1] = Ekin; out[2] = Efr; out[3] = Eel + Ekin + Efr;
}

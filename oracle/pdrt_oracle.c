/*
 * pdrt_oracle.c — float64 CPU ORACLE for the PyDoseRT dose hot path.
 *
 * TEST INFRASTRUCTURE ONLY.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may call this.  It shares no code, header,
 * table or constant generator with the CUDA path in paper_2512_18863_b200/csrc/.
 *
 * It follows the paper (arxiv 2512.18863, /root/reference/PAPER.md) step by step in
 * the paper's order, in float64, with dense plain loops.  Where the paper is silent
 * the readings G1..G22 of SURVEY.md §8(c) / DESIGN.md §3 are taken; each function
 * names the passage and the reading it follows.  The only liberties taken are ones
 * that cannot change a result: products with an exactly-zero fluence are skipped in
 * the slice convolution (a bounding box of the non-zero inputs), and independent
 * outer loops carry an OpenMP pragma.
 *
 * Parity pins (tests/test_oracle_pins.py): P1..P12 of SURVEY.md §8(c).
 * Parity UNPINNED (stated in DESIGN.md): the functional form and coefficients of the
 * pencil kernel K(r;z) (ref [17] of the paper is not available: the (A,a,B,b)(z)
 * tables are inputs), and the head-scatter / off-axis forms (words only in the paper).
 *
 * Layouts: patient volumes [nz][ny][nx] (x fastest); beam volumes [Nw][Nv][Nu]
 * (u fastest); fluence maps [Nvf][Nuf]; leaves [2][Np] (bank 0 = left l_i, bank 1 =
 * right r_i); jaws [4] = x1,x2 (along u), y1,y2 (along v).  Millimetres, degrees.
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>

typedef struct {
    int nx, ny, nz;
    double sx, sy, sz;      /* voxel spacing [mm]                 */
    double ox, oy, oz;      /* centre of voxel (0,0,0) [mm]       */
    double iso[3];          /* isocentre [mm], patient frame      */
} orc_grid;

typedef struct {
    double sid;                                   /* source-isocentre distance [mm]              */
    int n_pairs; const double *leaf_bounds;       /* n_pairs+1 leaf boundaries along v, ascending */
    int flu_nu, flu_nv; double flu_du, flu_dv;    /* fluence map size and pixel                  */
    double tau;                                   /* MLC transmission                            */
    double fwhm_mlc, fwhm_jaw;                    /* source penumbra FWHM along u / v; 0 = off   */
    int n_hs; const double *hs_amp, *hs_sigma;    /* head-scatter Gaussians; n_hs = 0 = off      */
    int n_oar; double oar_dr; const double *oar;  /* radial off-axis table; n_oar = 0 = off      */
    int n_z; double dz;                           /* kernel parameter table over radiological depth */
    const double *kA, *ka, *kB, *kb;              /* K(r;z) = (A e^{-a r} + B e^{-b r}) / r      */
    int kernel_size;                              /* odd                                         */
    double cal;                                   /* global dose scale                           */
    int beam_nu, beam_nw; double beam_du, beam_dw, beam_wmin;   /* beam grid (explicit, no defaults) */
    double ray_step;                              /* ray-march step [mm]                         */
} orc_model;

#define ORC_PI 3.14159265358979323846

/* ------------------------------------------------------------------ geometry (G1, G2) */
/* Gantry angle phi: u^ = (cos, sin, 0), w^ = (-sin, cos, 0), v^ = (0,0,1);
 * source = iso - SID w^.  Rotation about the isocentre, about patient z only. */
static void gantry_axes(double gantry_deg, double *c, double *s)
{
    double phi = gantry_deg * ORC_PI / 180.0;
    *c = cos(phi);
    *s = sin(phi);
}
static double beam_u(const orc_model *m, int i) { return (i - 0.5 * (m->beam_nu - 1)) * m->beam_du; }
static double beam_w(const orc_model *m, int k) { return m->beam_wmin + k * m->beam_dw; }
static double beam_v(const orc_grid *g, int j) { return g->oz + j * g->sz - g->iso[2]; }
static double flu_u(const orc_model *m, int a) { return (a - 0.5 * (m->flu_nu - 1)) * m->flu_du; }
static double flu_v(const orc_model *m, int b) { return (b - 0.5 * (m->flu_nv - 1)) * m->flu_dv; }

/* ------------------------------------------------------------------ O1: Eq. 4 */
/* PAPER.md:105-107, Eq. 4: fractional overlap of the opening [lo,hi] with the pixel
 * centred at c of width D:  f = max(0, min(hi, c+D/2) - max(lo, c-D/2)) / D.       */
double orc_ov(double c, double D, double lo, double hi)
{
    double a = fmin(hi, c + 0.5 * D) - fmax(lo, c - 0.5 * D);
    return a > 0.0 ? a / D : 0.0;
}
/* Derivatives of Eq. 4 ("stable subgradients"; reading G9: half-open
 * intervals, the derivative of max(0,x) at x = 0 is taken as 1 so a closed pair can open):
 *   d ov/d hi = (1/D) [c-D/2 <= hi < c+D/2] [hi >= max(lo, c-D/2)]
 *   d ov/d lo = -(1/D) [c-D/2 < lo <= c+D/2] [lo <= min(hi, c+D/2)]                  */
double orc_dov_dhi(double c, double D, double lo, double hi)
{
    double pl = c - 0.5 * D, pr = c + 0.5 * D;
    return (pl <= hi && hi < pr && hi >= fmax(lo, pl)) ? 1.0 / D : 0.0;
}
double orc_dov_dlo(double c, double D, double lo, double hi)
{
    double pl = c - 0.5 * D, pr = c + 0.5 * D;
    return (pl < lo && lo <= pr && lo <= fmin(hi, pr)) ? -1.0 / D : 0.0;
}

/* ------------------------------------------------------------------ O3: Gaussian taps */
/* PAPER.md:114 (source penumbra as Gaussian convolutions), reading G13:
 * taps g[t] ∝ exp(-(t D)^2 / 2 sigma^2), t = -T..T, T = ceil(3 sigma / D), sum g = 1;
 * sigma = 0 => identity (T = 0).  Returns T; g must hold 2T+1 values (T <= 64).    */
int orc_gauss_taps(double sigma, double D, double *g)
{
    if (!(sigma > 0.0)) { g[0] = 1.0; return 0; }
    int T = (int)ceil(3.0 * sigma / D);
    double sum = 0.0;
    for (int t = -T; t <= T; ++t) {
        g[t + T] = exp(-(t * D) * (t * D) / (2.0 * sigma * sigma));
        sum += g[t + T];
    }
    for (int t = 0; t <= 2 * T; ++t) g[t] /= sum;
    return T;
}
/* 1-D convolution along one axis of an [nv][nu] map, zero padding (G13). axis 0 = u, 1 = v. */
void orc_blur_axis(const double *in, double *out, int nu, int nv, int axis, int T, const double *g)
{
    for (int b = 0; b < nv; ++b)
        for (int a = 0; a < nu; ++a) {
            double s = 0.0;
            for (int t = -T; t <= T; ++t) {
                int aa = a + (axis == 0 ? t : 0), bb = b + (axis == 1 ? t : 0);
                if (aa < 0 || aa >= nu || bb < 0 || bb >= nv) continue;
                s += g[t + T] * in[bb * nu + aa];
            }
            out[b * nu + a] = s;
        }
}
/* Transpose of orc_blur_axis, written as the scatter that mirrors the loop above. */
void orc_blur_axis_T(const double *gout, double *gin, int nu, int nv, int axis, int T, const double *g)
{
    memset(gin, 0, sizeof(double) * (size_t)nu * nv);
    for (int b = 0; b < nv; ++b)
        for (int a = 0; a < nu; ++a)
            for (int t = -T; t <= T; ++t) {
                int aa = a + (axis == 0 ? t : 0), bb = b + (axis == 1 ? t : 0);
                if (aa < 0 || aa >= nu || bb < 0 || bb >= nv) continue;
                gin[bb * nu + aa] += g[t + T] * gout[b * nu + a];
            }
}

/* O5: radial off-axis factor, reading G14: linear interpolation of a radial
 * table with spacing oar_dr, clamped at the last entry; n_oar = 0 => 1.              */
static double oar_factor(const orc_model *m, double r)
{
    if (m->n_oar <= 0) return 1.0;
    double t = r / m->oar_dr;
    int n0 = (int)floor(t);
    if (n0 >= m->n_oar - 1) return m->oar[m->n_oar - 1];
    double f = t - n0;
    return (1.0 - f) * m->oar[n0] + f * m->oar[n0 + 1];
}

#define FWHM_TO_SIGMA 2.354820045

/* ------------------------------------------------------------------ O1..O5: fluence map */
/* PAPER.md:103-119 (FluenceMapLayer).  A, J, Phi0 may be NULL.  All maps [Nvf][Nuf].
 *  O1 (Eq. 4, G10): A[b][a] = sum_i ov(vf_b,Dv; vb_i,vb_{i+1}) * ov(uf_a,Du; l_i,r_i)
 *  O2 (:109 jaws "analogous masking", :113 transmission; G11, G12):
 *       J[b][a] = ov(uf_a,Du;x1,x2) * ov(vf_b,Dv;y1,y2);  Phi0 = J * (tau + (1-tau) A)
 *  O3 (:114, G13): Phi1 = G_v(sigma_jaw) * (G_u(sigma_mlc) * Phi0)
 *  O4 (:115, G14): Phi2 = Phi1 + sum_q amp_q * G_u(sigma_q) * G_v(sigma_q) * Phi0
 *  O5 (:116, G14): Phimap = Phi2 * OAR(r)                                              */
void orc_fluence(const orc_model *m, const double *leaves, const double *jaws,
                 double *A_out, double *J_out, double *Phi0_out, double *Phimap)
{
    const int nu = m->flu_nu, nv = m->flu_nv, np = m->n_pairs;
    const size_t n = (size_t)nu * nv;
    double *A = calloc(n, sizeof(double)), *J = calloc(n, sizeof(double));
    double *P0 = calloc(n, sizeof(double)), *t1 = calloc(n, sizeof(double)), *t2 = calloc(n, sizeof(double));
    double g[129];
    for (int b = 0; b < nv; ++b)
        for (int a = 0; a < nu; ++a) {
            double uf = flu_u(m, a), vf = flu_v(m, b), s = 0.0;
            for (int i = 0; i < np; ++i)
                s += orc_ov(vf, m->flu_dv, m->leaf_bounds[i], m->leaf_bounds[i + 1]) *
                     orc_ov(uf, m->flu_du, leaves[i], leaves[np + i]);
            A[b * nu + a] = s;
            J[b * nu + a] = orc_ov(uf, m->flu_du, jaws[0], jaws[1]) * orc_ov(vf, m->flu_dv, jaws[2], jaws[3]);
            P0[b * nu + a] = J[b * nu + a] * (m->tau + (1.0 - m->tau) * s);
        }
    int T = orc_gauss_taps(m->fwhm_mlc / FWHM_TO_SIGMA, m->flu_du, g);
    orc_blur_axis(P0, t1, nu, nv, 0, T, g);
    T = orc_gauss_taps(m->fwhm_jaw / FWHM_TO_SIGMA, m->flu_dv, g);
    orc_blur_axis(t1, Phimap, nu, nv, 1, T, g);                       /* Phimap holds Phi1 */
    for (int q = 0; q < m->n_hs; ++q) {
        T = orc_gauss_taps(m->hs_sigma[q], m->flu_dv, g);
        orc_blur_axis(P0, t1, nu, nv, 1, T, g);
        T = orc_gauss_taps(m->hs_sigma[q], m->flu_du, g);
        orc_blur_axis(t1, t2, nu, nv, 0, T, g);
        for (size_t e = 0; e < n; ++e) Phimap[e] += m->hs_amp[q] * t2[e];  /* -> Phi2 */
    }
    for (int b = 0; b < nv; ++b)
        for (int a = 0; a < nu; ++a) {
            double uf = flu_u(m, a), vf = flu_v(m, b);
            Phimap[b * nu + a] *= oar_factor(m, sqrt(uf * uf + vf * vf));
        }
    if (A_out) memcpy(A_out, A, n * sizeof(double));
    if (J_out) memcpy(J_out, J, n * sizeof(double));
    if (Phi0_out) memcpy(Phi0_out, P0, n * sizeof(double));
    free(A); free(J); free(P0); free(t1); free(t2);
}

/* O10 (fluence part): given gPhimap = d L / d Phimap, return d L / d leaves [2][Np] and
 * d L / d jaws [4] by walking orc_fluence backwards: OAR product, transposed Gaussians,
 * product rule for Phi0 = J (tau + (1-tau) A), Eq. 4 derivatives (G9).                  */
void orc_fluence_adjoint(const orc_model *m, const double *leaves, const double *jaws,
                         const double *gPhimap, double *d_leaves, double *d_jaws)
{
    const int nu = m->flu_nu, nv = m->flu_nv, np = m->n_pairs;
    const size_t n = (size_t)nu * nv;
    double *A = calloc(n, sizeof(double));
    double *g2 = calloc(n, sizeof(double)), *t1 = calloc(n, sizeof(double)), *t2 = calloc(n, sizeof(double));
    double *gP0 = calloc(n, sizeof(double));
    double g[129];
    for (int b = 0; b < nv; ++b)                                           /* recompute A */
        for (int a = 0; a < nu; ++a) {
            double uf = flu_u(m, a), vf = flu_v(m, b), s = 0.0;
            for (int i = 0; i < np; ++i)
                s += orc_ov(vf, m->flu_dv, m->leaf_bounds[i], m->leaf_bounds[i + 1]) *
                     orc_ov(uf, m->flu_du, leaves[i], leaves[np + i]);
            A[b * nu + a] = s;
        }
    for (int b = 0; b < nv; ++b)                                           /* O5 transposed */
        for (int a = 0; a < nu; ++a) {
            double uf = flu_u(m, a), vf = flu_v(m, b);
            g2[b * nu + a] = gPhimap[b * nu + a] * oar_factor(m, sqrt(uf * uf + vf * vf));
        }
    int T = orc_gauss_taps(m->fwhm_jaw / FWHM_TO_SIGMA, m->flu_dv, g);     /* O3 transposed */
    orc_blur_axis_T(g2, t1, nu, nv, 1, T, g);
    T = orc_gauss_taps(m->fwhm_mlc / FWHM_TO_SIGMA, m->flu_du, g);
    orc_blur_axis_T(t1, gP0, nu, nv, 0, T, g);
    for (int q = 0; q < m->n_hs; ++q) {                                    /* O4 transposed */
        T = orc_gauss_taps(m->hs_sigma[q], m->flu_du, g);
        orc_blur_axis_T(g2, t1, nu, nv, 0, T, g);
        T = orc_gauss_taps(m->hs_sigma[q], m->flu_dv, g);
        orc_blur_axis_T(t1, t2, nu, nv, 1, T, g);
        for (size_t e = 0; e < n; ++e) gP0[e] += m->hs_amp[q] * t2[e];
    }
    for (int i = 0; i < 2 * np; ++i) d_leaves[i] = 0.0;
    for (int i = 0; i < 4; ++i) d_jaws[i] = 0.0;
    for (int b = 0; b < nv; ++b)                                           /* O2, O1 */
        for (int a = 0; a < nu; ++a) {
            double uf = flu_u(m, a), vf = flu_v(m, b);
            double ju = orc_ov(uf, m->flu_du, jaws[0], jaws[1]), jv = orc_ov(vf, m->flu_dv, jaws[2], jaws[3]);
            double gJ = gP0[b * nu + a] * (m->tau + (1.0 - m->tau) * A[b * nu + a]);
            double gA = gP0[b * nu + a] * ju * jv * (1.0 - m->tau);
            d_jaws[0] += gJ * orc_dov_dlo(uf, m->flu_du, jaws[0], jaws[1]) * jv;
            d_jaws[1] += gJ * orc_dov_dhi(uf, m->flu_du, jaws[0], jaws[1]) * jv;
            d_jaws[2] += gJ * ju * orc_dov_dlo(vf, m->flu_dv, jaws[2], jaws[3]);
            d_jaws[3] += gJ * ju * orc_dov_dhi(vf, m->flu_dv, jaws[2], jaws[3]);
            for (int i = 0; i < np; ++i) {
                double ovv = orc_ov(vf, m->flu_dv, m->leaf_bounds[i], m->leaf_bounds[i + 1]);
                if (ovv == 0.0) continue;
                d_leaves[i] += gA * ovv * orc_dov_dlo(uf, m->flu_du, leaves[i], leaves[np + i]);
                d_leaves[np + i] += gA * ovv * orc_dov_dhi(uf, m->flu_du, leaves[i], leaves[np + i]);
            }
        }
    free(A); free(g2); free(t1); free(t2); free(gP0);
}

/* ------------------------------------------------------------------ O6: Eq. 7 */
/* Relative electron density at a point (G8): 0 outside the grid's physical box
 * [o - s/2, o + (N - 1/2) s] (closed), else trilinear with indices clamped to the edge. */
static double density_at(const orc_grid *g, const float *rho, double px, double py, double pz)
{
    const double P[3] = { px, py, pz };
    const double o[3] = { g->ox, g->oy, g->oz }, s[3] = { g->sx, g->sy, g->sz };
    const int N[3] = { g->nx, g->ny, g->nz };
    int i0[3], i1[3];
    double t[3];
    for (int d = 0; d < 3; ++d) {
        if (P[d] < o[d] - 0.5 * s[d] || P[d] > o[d] + (N[d] - 0.5) * s[d]) return 0.0;
        double f = (P[d] - o[d]) / s[d];
        int fl = (int)floor(f);
        t[d] = f - fl;
        i0[d] = fl < 0 ? 0 : (fl > N[d] - 1 ? N[d] - 1 : fl);
        i1[d] = fl + 1 < 0 ? 0 : (fl + 1 > N[d] - 1 ? N[d] - 1 : fl + 1);
    }
    double acc = 0.0;
    for (int c = 0; c < 8; ++c) {
        int ix = (c & 1) ? i1[0] : i0[0], iy = (c & 2) ? i1[1] : i0[1], iz = (c & 4) ? i1[2] : i0[2];
        double wx = (c & 1) ? t[0] : 1.0 - t[0], wy = (c & 2) ? t[1] : 1.0 - t[1], wz = (c & 4) ? t[2] : 1.0 - t[2];
        acc += wx * wy * wz * (double)rho[((size_t)iz * g->ny + iy) * g->nx + ix];
    }
    return acc;
}
/* PAPER.md:137-141, Eq. 7 (central-axis ray, one per gantry angle; G7), "cumulative
 * summation over uniformly sampled points" with reading G8:
 *   rho_m = rho(source + (m + 1/2) ds w^),  Z_0 = 0,  Z_{m+1} = Z_m + rho_m ds,
 *   slice k at distance SID + w_k:  q = (SID + w_k)/ds, m0 = floor(q),
 *   z_k = Z_{m0} + (q - m0) rho_{m0} ds.                                              */
void orc_radiological_depth(const orc_grid *g, const float *rho, const orc_model *m,
                            double gantry_deg, double *z)
{
    double c, s;
    gantry_axes(gantry_deg, &c, &s);
    const double wx = -s, wy = c;                        /* w^ */
    const double srcx = g->iso[0] - m->sid * wx, srcy = g->iso[1] - m->sid * wy, srcz = g->iso[2];
    const double ds = m->ray_step;
    double dmax = m->sid + beam_w(m, m->beam_nw - 1);
    int M = dmax > 0 ? (int)floor(dmax / ds) + 2 : 1;
    double *Z = malloc(sizeof(double) * (M + 1)), *r = malloc(sizeof(double) * (M + 1));
    Z[0] = 0.0;
    for (int mm = 0; mm < M; ++mm) {
        double t = (mm + 0.5) * ds;
        r[mm] = density_at(g, rho, srcx + t * wx, srcy + t * wy, srcz);
        Z[mm + 1] = Z[mm] + r[mm] * ds;
    }
    for (int k = 0; k < m->beam_nw; ++k) {
        double q = (m->sid + beam_w(m, k)) / ds;
        if (q <= 0.0) { z[k] = 0.0; continue; }
        int m0 = (int)floor(q);
        z[k] = Z[m0] + (q - m0) * r[m0] * ds;
    }
    free(Z); free(r);
}

/* ------------------------------------------------------------------ O7: pencil kernels */
/* PAPER.md:147 (radially symmetric K(r;z), depth-dependent amplitude and width), readings
 * G3 (two exponentials over r, parameters tabulated at z = n dz), G4 (pixel integration by
 * 8x8 midpoint sub-sampling, no renormalisation), G6 (depth dose carried by A(z), B(z)).
 * W_tab[n][dj][di] = (du dv / 64) * sum over the 8x8 sub-samples of pixel (di,dj) of K.   */
void orc_kernel_table(const orc_model *m, double dv, double *W_tab)
{
    const int k = m->kernel_size, c = (k - 1) / 2;
    const double du = m->beam_du;
    for (int n = 0; n < m->n_z; ++n)
        for (int dj = 0; dj < k; ++dj)
            for (int di = 0; di < k; ++di) {
                double s = 0.0;
                for (int sj = 0; sj < 8; ++sj)
                    for (int si = 0; si < 8; ++si) {
                        double x = ((di - c) + ((si + 0.5) / 8.0 - 0.5)) * du;
                        double y = ((dj - c) + ((sj + 0.5) / 8.0 - 0.5)) * dv;
                        double r = sqrt(x * x + y * y);
                        s += (m->kA[n] * exp(-m->ka[n] * r) + m->kB[n] * exp(-m->kb[n] * r)) / r;
                    }
                W_tab[((size_t)n * k + dj) * k + di] = s * du * dv / 64.0;
            }
}
/* Slice kernel at radiological depth z (G5: linear in z between table nodes):
 * t = z/dz, n0 = clamp(floor t, 0, n_z-2), W = (1-f) W_tab[n0] + f W_tab[n0+1], f = clamp(t-n0,0,1). */
void orc_slice_kernel(const orc_model *m, const double *W_tab, double z, double *W)
{
    const int k = m->kernel_size;
    double t = z / m->dz;
    int n0 = (int)floor(t);
    if (n0 < 0) n0 = 0;
    if (n0 > m->n_z - 2) n0 = m->n_z - 2;
    double f = t - n0;
    if (f < 0.0) f = 0.0;
    if (f > 1.0) f = 1.0;
    for (int e = 0; e < k * k; ++e)
        W[e] = (1.0 - f) * W_tab[(size_t)n0 * k * k + e] + f * W_tab[(size_t)(n0 + 1) * k * k + e];
}

/* ------------------------------------------------------------------ O8: Eq. 5, 6, 8 */
/* Interpolation between sample centres of a [n1][n0] array at fractional index (f0,f1);
 * neighbours outside the array contribute 0 ("bilinear_0" of SURVEY.md §8(c)).          */
static double bilinear0(const double *a, int n0, int n1, double f0, double f1)
{
    int i0 = (int)floor(f0), i1 = (int)floor(f1);
    double t0 = f0 - i0, t1 = f1 - i1, acc = 0.0;
    for (int c = 0; c < 4; ++c) {
        int x = i0 + (c & 1), y = i1 + (c >> 1);
        if (x < 0 || x >= n0 || y < 0 || y >= n1) continue;
        acc += ((c & 1) ? t0 : 1.0 - t0) * ((c >> 1) ? t1 : 1.0 - t1) * a[(size_t)y * n0 + x];
    }
    return acc;
}
/* PAPER.md:125-133, Eq. 5-6 (FluenceVolumeLayer), reading G15 (d = SID + w, axial):
 * mag = SID/d;  Phivol[k][j][i] = mag^2 * bilinear_0(Phimap; mag u_i/Du + (Nuf-1)/2, mag v_j/Dv + (Nvf-1)/2). */
void orc_project(const orc_grid *g, const orc_model *m, const double *Phimap, double *Phivol)
{
    const int Nu = m->beam_nu, Nv = g->nz, Nw = m->beam_nw;
#pragma omp parallel for schedule(static)
    for (int k = 0; k < Nw; ++k) {
        double mag = m->sid / (m->sid + beam_w(m, k));
        for (int j = 0; j < Nv; ++j)
            for (int i = 0; i < Nu; ++i) {
                double fa = mag * beam_u(m, i) / m->flu_du + 0.5 * (m->flu_nu - 1);
                double fb = mag * beam_v(g, j) / m->flu_dv + 0.5 * (m->flu_nv - 1);
                Phivol[((size_t)k * Nv + j) * Nu + i] = mag * mag * bilinear0(Phimap, m->flu_nu, m->flu_nv, fa, fb);
            }
    }
}
/* Transpose of orc_project: gPhimap[pix] = sum over voxels of mag^2 * weight(voxel->pix) * H[voxel]. */
void orc_project_adjoint(const orc_grid *g, const orc_model *m, const double *H, double *gPhimap)
{
    const int Nu = m->beam_nu, Nv = g->nz, Nw = m->beam_nw, n0 = m->flu_nu, n1 = m->flu_nv;
    memset(gPhimap, 0, sizeof(double) * (size_t)n0 * n1);
    for (int k = 0; k < Nw; ++k) {
        double mag = m->sid / (m->sid + beam_w(m, k));
        for (int j = 0; j < Nv; ++j)
            for (int i = 0; i < Nu; ++i) {
                double h = H[((size_t)k * Nv + j) * Nu + i];
                if (h == 0.0) continue;
                double fa = mag * beam_u(m, i) / m->flu_du + 0.5 * (n0 - 1);
                double fb = mag * beam_v(g, j) / m->flu_dv + 0.5 * (n1 - 1);
                int i0 = (int)floor(fa), i1 = (int)floor(fb);
                double t0 = fa - i0, t1 = fb - i1;
                for (int c = 0; c < 4; ++c) {
                    int x = i0 + (c & 1), y = i1 + (c >> 1);
                    if (x < 0 || x >= n0 || y < 0 || y >= n1) continue;
                    gPhimap[(size_t)y * n0 + x] += mag * mag * ((c & 1) ? t0 : 1.0 - t0) * ((c >> 1) ? t1 : 1.0 - t1) * h;
                }
            }
    }
}
/* PAPER.md:153-158, Eq. 8 (BeamWiseConvolutionLayer): each depth slice convolved with its own
 * kernel, zero-padded "same":  D[k][j][i] = sum_{dj,di} W_k[dj][di] Phivol[k][j+dj-c][i+di-c].
 * Inputs that are exactly zero are skipped through the bounding box of the non-zero inputs. */
void orc_convolve(const orc_grid *g, const orc_model *m, const double *W_tab, const double *z,
                  const double *Phivol, double *D)
{
    const int Nu = m->beam_nu, Nv = g->nz, Nw = m->beam_nw, K = m->kernel_size, c = (K - 1) / 2;
#pragma omp parallel for schedule(dynamic, 1)
    for (int k = 0; k < Nw; ++k) {
        double *W = malloc(sizeof(double) * K * K);
        orc_slice_kernel(m, W_tab, z[k], W);
        const double *P = Phivol + (size_t)k * Nv * Nu;
        int i_lo = Nu, i_hi = -1, j_lo = Nv, j_hi = -1;
        for (int j = 0; j < Nv; ++j)
            for (int i = 0; i < Nu; ++i)
                if (P[(size_t)j * Nu + i] != 0.0) {
                    if (i < i_lo) i_lo = i;
                    if (i > i_hi) i_hi = i;
                    if (j < j_lo) j_lo = j;
                    if (j > j_hi) j_hi = j;
                }
        for (int j = 0; j < Nv; ++j)
            for (int i = 0; i < Nu; ++i) {
                double s = 0.0;
                for (int dj = 0; dj < K; ++dj) {
                    int jj = j + dj - c;
                    if (jj < 0 || jj >= Nv || jj < j_lo || jj > j_hi) continue;
                    for (int di = 0; di < K; ++di) {
                        int ii = i + di - c;
                        if (ii < 0 || ii >= Nu || ii < i_lo || ii > i_hi) continue;
                        s += W[dj * K + di] * P[(size_t)jj * Nu + ii];
                    }
                }
                D[((size_t)k * Nv + j) * Nu + i] = s;
            }
        free(W);
    }
}
/* Transpose of orc_convolve (dense, no skipping): H[k][jj][ii] = sum over outputs (j,i) that read
 * input (jj,ii):  H[jj][ii] += W[dj][di] G[j][i]  with jj = j+dj-c, ii = i+di-c.                  */
void orc_convolve_adjoint(const orc_grid *g, const orc_model *m, const double *W_tab, const double *z,
                          const double *G, double *H)
{
    const int Nu = m->beam_nu, Nv = g->nz, Nw = m->beam_nw, K = m->kernel_size, c = (K - 1) / 2;
#pragma omp parallel for schedule(dynamic, 1)
    for (int k = 0; k < Nw; ++k) {
        double *W = malloc(sizeof(double) * K * K);
        orc_slice_kernel(m, W_tab, z[k], W);
        const double *Gk = G + (size_t)k * Nv * Nu;
        double *Hk = H + (size_t)k * Nv * Nu;
        memset(Hk, 0, sizeof(double) * (size_t)Nv * Nu);
        for (int j = 0; j < Nv; ++j)
            for (int i = 0; i < Nu; ++i) {
                double gv = Gk[(size_t)j * Nu + i];
                if (gv == 0.0) continue;
                for (int dj = 0; dj < K; ++dj) {
                    int jj = j + dj - c;
                    if (jj < 0 || jj >= Nv) continue;
                    for (int di = 0; di < K; ++di) {
                        int ii = i + di - c;
                        if (ii < 0 || ii >= Nu) continue;
                        Hk[(size_t)jj * Nu + ii] += W[dj * K + di] * gv;
                    }
                }
            }
        free(W);
    }
}

/* ------------------------------------------------------------------ O9: Eq. 9 */
/* PAPER.md:162 (BeamRotationLayer: the inverse rotation maps patient-frame positions to beam-frame
 * sampling locations; readings G1, G2: rotation about the isocentre and patient z only, so the
 * trilinear interpolation is bilinear in the (u,w) plane of the matching z slice; zero outside the
 * beam grid) and :164-168, Eq. 9:  dose[p] += scale * bilinear_0(D_b[.][z(p)][.]; fu, fw).        */
void orc_resample_add(const orc_grid *g, const orc_model *m, double gantry_deg, double scale,
                      const double *Db, double *dose)
{
    const int Nu = m->beam_nu, Nv = g->nz, Nw = m->beam_nw;
    double c, s;
    gantry_axes(gantry_deg, &c, &s);
#pragma omp parallel for schedule(static)
    for (int kz = 0; kz < g->nz; ++kz)
        for (int jy = 0; jy < g->ny; ++jy)
            for (int ix = 0; ix < g->nx; ++ix) {
                double dx = g->ox + ix * g->sx - g->iso[0], dy = g->oy + jy * g->sy - g->iso[1];
                double u = c * dx + s * dy, w = -s * dx + c * dy;
                double fu = u / m->beam_du + 0.5 * (Nu - 1), fw = (w - m->beam_wmin) / m->beam_dw;
                int i0 = (int)floor(fu), k0 = (int)floor(fw);
                double tu = fu - i0, tw = fw - k0, acc = 0.0;
                for (int q = 0; q < 4; ++q) {
                    int i = i0 + (q & 1), k = k0 + (q >> 1);
                    if (i < 0 || i >= Nu || k < 0 || k >= Nw) continue;
                    acc += ((q & 1) ? tu : 1.0 - tu) * ((q >> 1) ? tw : 1.0 - tw) * Db[((size_t)k * Nv + kz) * Nu + i];
                }
                dose[((size_t)kz * g->ny + jy) * g->nx + ix] += scale * acc;
            }
}
/* Transpose of orc_resample_add with scale = 1:  G[k][z][i] += weight * gdose[p]. */
void orc_resample_adjoint(const orc_grid *g, const orc_model *m, double gantry_deg,
                          const float *gdose, double *G)
{
    const int Nu = m->beam_nu, Nv = g->nz, Nw = m->beam_nw;
    double c, s;
    gantry_axes(gantry_deg, &c, &s);
    memset(G, 0, sizeof(double) * (size_t)Nu * Nv * Nw);
#pragma omp parallel for schedule(static)
    for (int kz = 0; kz < g->nz; ++kz)          /* slices write disjoint G[.][kz][.] */
        for (int jy = 0; jy < g->ny; ++jy)
            for (int ix = 0; ix < g->nx; ++ix) {
                double gv = (double)gdose[((size_t)kz * g->ny + jy) * g->nx + ix];
                if (gv == 0.0) continue;
                double dx = g->ox + ix * g->sx - g->iso[0], dy = g->oy + jy * g->sy - g->iso[1];
                double u = c * dx + s * dy, w = -s * dx + c * dy;
                double fu = u / m->beam_du + 0.5 * (Nu - 1), fw = (w - m->beam_wmin) / m->beam_dw;
                int i0 = (int)floor(fu), k0 = (int)floor(fw);
                double tu = fu - i0, tw = fw - k0;
                for (int q = 0; q < 4; ++q) {
                    int i = i0 + (q & 1), k = k0 + (q >> 1);
                    if (i < 0 || i >= Nu || k < 0 || k >= Nw) continue;
                    G[((size_t)k * Nv + kz) * Nu + i] += ((q & 1) ? tu : 1.0 - tu) * ((q >> 1) ? tw : 1.0 - tw) * gv;
                }
            }
}

/* ------------------------------------------------------------------ whole path */
/* One control point, beam frame:  D_b = conv(project(fluence(theta_b)); kernels at z_rad(phi_b)). */
void orc_beam_dose(const orc_grid *g, const orc_model *m, const float *rho, const double *W_tab,
                   const double *leaves, const double *jaws, double gantry_deg, double *Db)
{
    const size_t nb = (size_t)m->beam_nu * g->nz * m->beam_nw;
    double *Phimap = malloc(sizeof(double) * (size_t)m->flu_nu * m->flu_nv);
    double *Phivol = malloc(sizeof(double) * nb), *z = malloc(sizeof(double) * m->beam_nw);
    orc_fluence(m, leaves, jaws, NULL, NULL, NULL, Phimap);
    orc_radiological_depth(g, rho, m, gantry_deg, z);
    orc_project(g, m, Phimap, Phivol);
    orc_convolve(g, m, W_tab, z, Phivol, Db);
    free(Phimap); free(Phivol); free(z);
}
/* PAPER.md:164-168, Eq. 9:  D_total = cal * sum_b MU_b * R_b D_b   (cal: :178 energy scaling factor).
 * W_tab is the table of orc_kernel_table for m->kernel_size (the caller builds it once per kernel size). */
void orc_dose(const orc_grid *g, const orc_model *m, const float *rho, const double *W_tab, int n_cp,
              const double *leaves, const double *jaws, const double *gantry_deg, const double *mu,
              double *dose)
{
    const size_t nb = (size_t)m->beam_nu * g->nz * m->beam_nw, np = (size_t)g->nx * g->ny * g->nz;
    double *Db = malloc(sizeof(double) * nb);
    memset(dose, 0, sizeof(double) * np);
    for (int b = 0; b < n_cp; ++b) {
        orc_beam_dose(g, m, rho, W_tab, leaves + (size_t)b * 2 * m->n_pairs, jaws + (size_t)b * 4, gantry_deg[b], Db);
        orc_resample_add(g, m, gantry_deg[b], m->cal * mu[b], Db, dose);
    }
    free(Db);
}
/* O10: dL/d(leaves, jaws, MU) from gdose = dL/dDose, by the transposes in reverse order.
 * Everything after the fluence map is linear and MU is a scalar factor, so
 *   d_mu_b = cal <R_b^T g, D_b> = cal <gPhimap_b, Phimap_b>,  gPhimap_b = P^T C^T R_b^T g,
 *   d(leaves,jaws)_b = cal MU_b * (d Phimap_b / d theta)^T gPhimap_b.
 * Radiological depth and kernels carry no gradient.                   */
void orc_dose_backward(const orc_grid *g, const orc_model *m, const float *rho, const double *W_tab, int n_cp,
                       const double *leaves, const double *jaws, const double *gantry_deg, const double *mu,
                       const float *gdose, double *d_leaves, double *d_jaws, double *d_mu)
{
    const size_t nb = (size_t)m->beam_nu * g->nz * m->beam_nw, nf = (size_t)m->flu_nu * m->flu_nv;
    const int np = m->n_pairs;
    double *G = malloc(sizeof(double) * nb), *H = malloc(sizeof(double) * nb), *z = malloc(sizeof(double) * m->beam_nw);
    double *Phimap = malloc(sizeof(double) * nf), *gPhimap = malloc(sizeof(double) * nf);
    for (int b = 0; b < n_cp; ++b) {
        const double *lv = leaves + (size_t)b * 2 * np, *jw = jaws + (size_t)b * 4;
        orc_fluence(m, lv, jw, NULL, NULL, NULL, Phimap);
        orc_radiological_depth(g, rho, m, gantry_deg[b], z);
        orc_resample_adjoint(g, m, gantry_deg[b], gdose, G);
        orc_convolve_adjoint(g, m, W_tab, z, G, H);
        orc_project_adjoint(g, m, H, gPhimap);
        double dot = 0.0;
        for (size_t e = 0; e < nf; ++e) dot += Phimap[e] * gPhimap[e];
        d_mu[b] = m->cal * dot;
        orc_fluence_adjoint(m, lv, jw, gPhimap, d_leaves + (size_t)b * 2 * np, d_jaws + (size_t)b * 4);
        for (int e = 0; e < 2 * np; ++e) d_leaves[(size_t)b * 2 * np + e] *= m->cal * mu[b];
        for (int e = 0; e < 4; ++e) d_jaws[(size_t)b * 4 + e] *= m->cal * mu[b];
    }
    free(G); free(H); free(z); free(Phimap); free(gPhimap);
}

/* Dose at selected patient voxels only (ijk triplets = x,y,z indices): the same definitions as
 * orc_dose, evaluated one output at a time, so that full-size workloads can be spot-checked.
 * For each point and control point: the 4 beam voxels of the bilinear stencil, each the direct
 * sum of Eq. 8 over the k x k window of projected fluence (Eq. 5-6).                           */
void orc_dose_at(const orc_grid *g, const orc_model *m, const float *rho, const double *W_tab, int n_cp,
                 const double *leaves, const double *jaws, const double *gantry_deg, const double *mu,
                 int n_pts, const int *ijk, double *out)
{
    const int Nu = m->beam_nu, Nv = g->nz, Nw = m->beam_nw, K = m->kernel_size, c = (K - 1) / 2;
    for (int p = 0; p < n_pts; ++p) out[p] = 0.0;
#pragma omp parallel
    {
        double *Phimap = malloc(sizeof(double) * (size_t)m->flu_nu * m->flu_nv);
        double *z = malloc(sizeof(double) * Nw), *W = malloc(sizeof(double) * K * K);
        double *part = calloc(n_pts, sizeof(double));
#pragma omp for schedule(dynamic, 1)
        for (int b = 0; b < n_cp; ++b) {
            double cs, sn;
            gantry_axes(gantry_deg[b], &cs, &sn);
            orc_fluence(m, leaves + (size_t)b * 2 * m->n_pairs, jaws + (size_t)b * 4, NULL, NULL, NULL, Phimap);
            orc_radiological_depth(g, rho, m, gantry_deg[b], z);
            for (int p = 0; p < n_pts; ++p) {
                int ix = ijk[3 * p], jy = ijk[3 * p + 1], kz = ijk[3 * p + 2];
                double dx = g->ox + ix * g->sx - g->iso[0], dy = g->oy + jy * g->sy - g->iso[1];
                double u = cs * dx + sn * dy, w = -sn * dx + cs * dy;
                double fu = u / m->beam_du + 0.5 * (Nu - 1), fw = (w - m->beam_wmin) / m->beam_dw;
                int i0 = (int)floor(fu), k0 = (int)floor(fw);
                double tu = fu - i0, tw = fw - k0, acc = 0.0;
                for (int q = 0; q < 4; ++q) {
                    int i = i0 + (q & 1), k = k0 + (q >> 1);
                    if (i < 0 || i >= Nu || k < 0 || k >= Nw) continue;
                    double mag = m->sid / (m->sid + beam_w(m, k)), d = 0.0;
                    orc_slice_kernel(m, W_tab, z[k], W);
                    for (int dj = 0; dj < K; ++dj) {
                        int jj = kz + dj - c;
                        if (jj < 0 || jj >= Nv) continue;
                        for (int di = 0; di < K; ++di) {
                            int ii = i + di - c;
                            if (ii < 0 || ii >= Nu) continue;
                            double fa = mag * beam_u(m, ii) / m->flu_du + 0.5 * (m->flu_nu - 1);
                            double fb = mag * beam_v(g, jj) / m->flu_dv + 0.5 * (m->flu_nv - 1);
                            d += W[dj * K + di] * mag * mag * bilinear0(Phimap, m->flu_nu, m->flu_nv, fa, fb);
                        }
                    }
                    acc += ((q & 1) ? tu : 1.0 - tu) * ((q >> 1) ? tw : 1.0 - tw) * d;
                }
                part[p] += m->cal * mu[b] * acc;
            }
        }
#pragma omp critical
        for (int p = 0; p < n_pts; ++p) out[p] += part[p];
        free(Phimap); free(z); free(W); free(part);
    }
}

#ifdef _OPENMP
#include <omp.h>
int orc_num_threads(void) { return omp_get_max_threads(); }
#else
int orc_num_threads(void) { return 1; }
#endif

/* ================================================================== planning loop */
/* PAPER.md:83-101, Eq. 1-3 (BeamValidationLayer).  For every opposing pair (p_a, p_b) — each leaf pair and the two jaw
 * pairs (x1,x2), (y1,y2):
 *   Eq. 1:  c = (p_a + p_b)/2,  w = p_b - p_a;   w >= w_min enforced,  c clamped to [-F, F];
 *   Eq. 2:  p_a^ = c - w/2,  p_b^ = c + w/2.
 * Monitor units are clamped to mu_eps > 0 (reading G16).  Limits: lim[0] = leaf w_min, lim[1] = leaf F,
 * lim[2] = jaw w_min, lim[3] = jaw-x F, lim[4] = jaw-y F, lim[5] = mu_eps.                                          */
static void validate_pair(double pa, double pb, double w_min, double F, double *qa, double *qb)
{
    double c = 0.5 * (pa + pb), w = pb - pa;
    if (w < w_min) w = w_min;
    if (c < -F) c = -F;
    if (c > F) c = F;
    *qa = c - 0.5 * w;
    *qb = c + 0.5 * w;
}
void orc_validate(int n_cp, int n_pairs, const double *lim, const double *leaves, const double *jaws, const double *mu,
                  double *leaves_out, double *jaws_out, double *mu_out)
{
    for (int b = 0; b < n_cp; ++b) {
        const double *lv = leaves + (size_t)b * 2 * n_pairs;
        double *lo = leaves_out + (size_t)b * 2 * n_pairs;
        for (int i = 0; i < n_pairs; ++i) validate_pair(lv[i], lv[n_pairs + i], lim[0], lim[1], &lo[i], &lo[n_pairs + i]);
        validate_pair(jaws[4 * b + 0], jaws[4 * b + 1], lim[2], lim[3], &jaws_out[4 * b + 0], &jaws_out[4 * b + 1]);
        validate_pair(jaws[4 * b + 2], jaws[4 * b + 3], lim[2], lim[4], &jaws_out[4 * b + 2], &jaws_out[4 * b + 3]);
        mu_out[b] = mu[b] < lim[5] ? lim[5] : mu[b];
    }
}
/* Transpose of the Jacobian of orc_validate at the raw parameters ("preserve gradients").  The map is
 * piecewise linear; reading G23: a clamp passes the gradient where its input lies inside the closed
 * interval, i.e. [w >= w_min], [-F <= c <= F], [mu >= mu_eps], and blocks it outside (the convention of a clamp in an
 * automatic-differentiation framework, which is what the paper's layer is built from).
 *   g_c^ = g_a^ + g_b^,  g_w^ = (g_b^ - g_a^)/2;   g_c = g_c^ [c in range],  g_w = g_w^ [w >= w_min];
 *   g_a = g_c/2 - g_w,  g_b = g_c/2 + g_w.                                                                          */
static void validate_pair_adjoint(double pa, double pb, double w_min, double F, double ga_hat, double gb_hat, double *ga, double *gb)
{
    double c = 0.5 * (pa + pb), w = pb - pa;
    double gc = ga_hat + gb_hat, gw = 0.5 * (gb_hat - ga_hat);
    if (!(c >= -F && c <= F)) gc = 0.0;
    if (!(w >= w_min)) gw = 0.0;
    *ga = 0.5 * gc - gw;
    *gb = 0.5 * gc + gw;
}
void orc_validate_adjoint(int n_cp, int n_pairs, const double *lim, const double *leaves, const double *jaws, const double *mu,
                          const double *g_leaves_hat, const double *g_jaws_hat, const double *g_mu_hat,
                          double *g_leaves, double *g_jaws, double *g_mu)
{
    for (int b = 0; b < n_cp; ++b) {
        const size_t o = (size_t)b * 2 * n_pairs;
        for (int i = 0; i < n_pairs; ++i)
            validate_pair_adjoint(leaves[o + i], leaves[o + n_pairs + i], lim[0], lim[1], g_leaves_hat[o + i], g_leaves_hat[o + n_pairs + i],
                                  &g_leaves[o + i], &g_leaves[o + n_pairs + i]);
        validate_pair_adjoint(jaws[4 * b], jaws[4 * b + 1], lim[2], lim[3], g_jaws_hat[4 * b], g_jaws_hat[4 * b + 1], &g_jaws[4 * b], &g_jaws[4 * b + 1]);
        validate_pair_adjoint(jaws[4 * b + 2], jaws[4 * b + 3], lim[2], lim[4], g_jaws_hat[4 * b + 2], g_jaws_hat[4 * b + 3], &g_jaws[4 * b + 2], &g_jaws[4 * b + 3]);
        g_mu[b] = mu[b] >= lim[5] ? g_mu_hat[b] : 0.0;
    }
}
/* PAPER.md:99, Eq. 3: minimum MU per control point from machine dynamics. */
double orc_mu_epsilon(double dose_rate_min, double delta_phi, double gantry_speed_max) { return dose_rate_min * delta_phi / gantry_speed_max; }

/* Weighted-sum objective over structures and its dose gradient.  PAPER.md:205-210, Eq. 10 is the case power = 1:
 *   L = sum_s lambda_s || D_s - p_s ||_1     (p_s = prescription of the target, 0 for organs at risk);
 * power = 2 is the quadratic objective BASELINE.json's configs c4/c5 name: L = sum_s lambda_s sum_{x in s} (D(x)-p_s)^2.
 * Structures may overlap: bits[x] has bit s set when voxel x belongs to structure s (s < 32).
 * g = dL/dD:  power 1: sum_s lambda_s sign(D - p_s) (sign(0) = 0, a valid subgradient);  power 2: sum_s 2 lambda_s (D - p_s). */
double orc_objective(size_t n_vox, const float *dose, const unsigned *bits, int n_struct, const double *lambda, const double *presc,
                     int power, float *g)
{
    double L = 0.0;
    for (size_t x = 0; x < n_vox; ++x) {
        double gx = 0.0;
        for (int s = 0; s < n_struct; ++s) {
            if (!((bits[x] >> s) & 1u)) continue;
            double d = (double)dose[x] - presc[s];
            if (power == 1) { L += lambda[s] * fabs(d); gx += lambda[s] * (d > 0.0 ? 1.0 : (d < 0.0 ? -1.0 : 0.0)); }
            else { L += lambda[s] * d * d; gx += 2.0 * lambda[s] * d; }
        }
        if (g) g[x] = (float)gx;
    }
    return L;
}

/* Jaws tracking the aperture (BASELINE.json configs[4] "jaws tracking the aperture"; recipe of SURVEY.md §8(d) c5): over
 * the pairs that are open by more than open_gap:  x1 = min l - margin, x2 = max r + margin, y1 / y2 = the v-extent of
 * those pairs (their leaf boundaries); when no pair is open, all pairs count as open.                               */
void orc_track_jaws(int n_cp, int n_pairs, const double *leaf_bounds, const double *leaves, double margin, double open_gap, double *jaws)
{
    for (int b = 0; b < n_cp; ++b) {
        const double *lv = leaves + (size_t)b * 2 * n_pairs;
        int any = 0;
        for (int i = 0; i < n_pairs; ++i) any |= (lv[n_pairs + i] - lv[i]) > open_gap;
        double x1 = 0, x2 = 0, y1 = 0, y2 = 0;
        int first = 1;
        for (int i = 0; i < n_pairs; ++i) {
            if (any && !((lv[n_pairs + i] - lv[i]) > open_gap)) continue;
            if (first) { x1 = lv[i]; x2 = lv[n_pairs + i]; y1 = leaf_bounds[i]; first = 0; }
            if (lv[i] < x1) x1 = lv[i];
            if (lv[n_pairs + i] > x2) x2 = lv[n_pairs + i];
            y2 = leaf_bounds[i + 1];
        }
        jaws[4 * b] = x1 - margin; jaws[4 * b + 1] = x2 + margin; jaws[4 * b + 2] = y1; jaws[4 * b + 3] = y2;
    }
}

/* Normalised-gradient step of the c5 planning loop: every leaf edge moves by at most step_leaf and
 * every MU by at most step_mu per iteration:  theta <- theta - step * g / max|g|, the maximum taken over the whole
 * group (all leaf edges of the arc; all MUs); a group whose gradient is identically zero does not move.             */
void orc_plan_step(int n_cp, int n_pairs, double step_leaf, double step_mu, const double *g_leaves, const double *g_mu,
                   double *leaves, double *mu)
{
    const size_t nl = (size_t)n_cp * 2 * n_pairs;
    double ml = 0.0, mm = 0.0;
    for (size_t e = 0; e < nl; ++e) if (fabs(g_leaves[e]) > ml) ml = fabs(g_leaves[e]);
    for (int b = 0; b < n_cp; ++b) if (fabs(g_mu[b]) > mm) mm = fabs(g_mu[b]);
    if (ml > 0.0) for (size_t e = 0; e < nl; ++e) leaves[e] -= step_leaf * g_leaves[e] / ml;
    if (mm > 0.0) for (int b = 0; b < n_cp; ++b) mu[b] -= step_mu * g_mu[b] / mm;
}

/* ================================================================== divergent radiological depth */
/* PAPER.md:137 traces ONE ray per gantry angle and names the consequence (:197, :357): reduced accuracy where the patient
 * surface is oblique to the beam.  This optional mode (reading G24) traces one diverging ray per fluence-map
 * pixel (a,b): from the source through (uf_a, vf_b) on the isocentre plane,
 *     P(t) = source + t * (w^ + (uf_a/SID) u^ + (vf_b/SID) v^),     t = distance travelled ALONG THE AXIS,
 * with the sampling rule of Eq. 7 / G8 in t (rho_m at t = (m + 1/2) ds, Z_{m+1} = Z_m + rho_m ds, linear within a step), so
 * that z_fan[k][b][a] is the radiological depth, measured along the axis direction, at which ray (a,b) crosses slice k.
 * Depth is counted per unit AXIAL distance: in a medium that is homogeneous across the beam every ray then reproduces the
 * central-axis profile exactly, and the mode reduces to the paper's.                                                     */
void orc_fan_depth(const orc_grid *g, const float *rho, const orc_model *m, double gantry_deg, double *z_fan)
{
    double c, s;
    gantry_axes(gantry_deg, &c, &s);
    const double ux = c, uy = s, wx = -s, wy = c;
    const double srcx = g->iso[0] - m->sid * wx, srcy = g->iso[1] - m->sid * wy, srcz = g->iso[2];
    const double ds = m->ray_step;
    const int Nw = m->beam_nw, nu = m->flu_nu, nv = m->flu_nv;
    double dmax = m->sid + beam_w(m, Nw - 1);
    int M = dmax > 0 ? (int)floor(dmax / ds) + 2 : 1;
#pragma omp parallel
    {
        double *Z = malloc(sizeof(double) * (M + 1)), *r = malloc(sizeof(double) * (M + 1));
#pragma omp for schedule(static)
        for (int b = 0; b < nv; ++b)
            for (int a = 0; a < nu; ++a) {
                const double tu = flu_u(m, a) / m->sid, tv = flu_v(m, b) / m->sid;
                const double dx = wx + tu * ux, dy = wy + tu * uy, dz = tv;
                Z[0] = 0.0;
                for (int mm = 0; mm < M; ++mm) {
                    double t = (mm + 0.5) * ds;
                    r[mm] = density_at(g, rho, srcx + t * dx, srcy + t * dy, srcz + t * dz);
                    Z[mm + 1] = Z[mm] + r[mm] * ds;
                }
                for (int k = 0; k < Nw; ++k) {
                    double q = (m->sid + beam_w(m, k)) / ds, zz = 0.0;
                    if (q > 0.0) { int m0 = (int)floor(q); zz = Z[m0] + (q - m0) * r[m0] * ds; }
                    z_fan[((size_t)k * nv + b) * nu + a] = zz;
                }
            }
        free(Z); free(r);
    }
}
/* Broad-beam depth term carried by the kernel amplitudes (reading G6): the plane integral of K(r;z),
 * T(z) = 2 pi (A(z)/a(z) + B(z)/b(z)), tabulated at the kernel table's nodes and interpolated linearly like the kernels (G5). */
double orc_depth_term(const orc_model *m, double z)
{
    double t = z / m->dz;
    int n0 = (int)floor(t);
    if (n0 < 0) n0 = 0;
    if (n0 > m->n_z - 2) n0 = m->n_z - 2;
    double f = t - n0;
    if (f < 0.0) f = 0.0;
    if (f > 1.0) f = 1.0;
    double T0 = 2.0 * ORC_PI * (m->kA[n0] / m->ka[n0] + m->kB[n0] / m->kb[n0]);
    double T1 = 2.0 * ORC_PI * (m->kA[n0 + 1] / m->ka[n0 + 1] + m->kB[n0 + 1] / m->kb[n0 + 1]);
    return (1.0 - f) * T0 + f * T1;
}
/* Depth factor at the ray nodes: F[k][b][a] = T(z_fan[k][b][a]) / T(z_cax[k]); 1 where T(z_cax[k]) <= 0 (the slice kernel
 * is zero there, so is the dose).  It weights the projected fluence (input side); the lateral kernel stays per slice.   */
void orc_fan_factor(const orc_grid *g, const orc_model *m, const double *z_fan, const double *z_cax, double *F)
{
    (void)g;
    const size_t nf = (size_t)m->flu_nu * m->flu_nv;
    for (int k = 0; k < m->beam_nw; ++k) {
        double Tc = orc_depth_term(m, z_cax[k]);
        for (size_t e = 0; e < nf; ++e) F[(size_t)k * nf + e] = Tc > 0.0 ? orc_depth_term(m, z_fan[(size_t)k * nf + e]) / Tc : 1.0;
    }
}
/* Interpolation between node centres with the indices clamped to the array (the depth factor exists beyond the map's edge). */
static double bilinear_clamp(const double *a, int n0, int n1, double f0, double f1)
{
    int i0 = (int)floor(f0), i1 = (int)floor(f1);
    double t0 = f0 - i0, t1 = f1 - i1, acc = 0.0;
    for (int c = 0; c < 4; ++c) {
        int x = i0 + (c & 1), y = i1 + (c >> 1);
        x = x < 0 ? 0 : (x > n0 - 1 ? n0 - 1 : x);
        y = y < 0 ? 0 : (y > n1 - 1 ? n1 - 1 : y);
        acc += ((c & 1) ? t0 : 1.0 - t0) * ((c >> 1) ? t1 : 1.0 - t1) * a[(size_t)y * n0 + x];
    }
    return acc;
}
/* Depth-weighted projection: Phivol'[k][j][i] = Phivol[k][j][i] * bilinear_clamp(F[k]; fa, fb) with (fa, fb) the sampling
 * position of Eq. 5 — the factor of the ray through the voxel, interpolated between the ray nodes.  `transpose` applies the
 * same diagonal weighting to H before orc_project_adjoint (the factor carries no gradient).                              */
void orc_apply_fan_factor(const orc_grid *g, const orc_model *m, const double *F, double *vol)
{
    const int Nu = m->beam_nu, Nv = g->nz, Nw = m->beam_nw;
    const size_t nf = (size_t)m->flu_nu * m->flu_nv;
#pragma omp parallel for schedule(static)
    for (int k = 0; k < Nw; ++k) {
        double mag = m->sid / (m->sid + beam_w(m, k));
        for (int j = 0; j < Nv; ++j)
            for (int i = 0; i < Nu; ++i) {
                double *p = &vol[((size_t)k * Nv + j) * Nu + i];
                if (*p == 0.0) continue;
                double fa = mag * beam_u(m, i) / m->flu_du + 0.5 * (m->flu_nu - 1);
                double fb = mag * beam_v(g, j) / m->flu_dv + 0.5 * (m->flu_nv - 1);
                *p *= bilinear_clamp(F + (size_t)k * nf, m->flu_nu, m->flu_nv, fa, fb);
            }
    }
}
/* Whole path in the divergent-depth mode: as orc_dose / orc_dose_backward with the projected fluence (resp. H) weighted. */
void orc_dose_fan(const orc_grid *g, const orc_model *m, const float *rho, const double *W_tab, int n_cp,
                  const double *leaves, const double *jaws, const double *gantry_deg, const double *mu, double *dose)
{
    const size_t nb = (size_t)m->beam_nu * g->nz * m->beam_nw, np = (size_t)g->nx * g->ny * g->nz;
    const size_t nf = (size_t)m->flu_nu * m->flu_nv;
    double *Db = malloc(sizeof(double) * nb), *Phivol = malloc(sizeof(double) * nb), *Phimap = malloc(sizeof(double) * nf);
    double *z = malloc(sizeof(double) * m->beam_nw), *zf = malloc(sizeof(double) * nf * m->beam_nw), *F = malloc(sizeof(double) * nf * m->beam_nw);
    memset(dose, 0, sizeof(double) * np);
    for (int b = 0; b < n_cp; ++b) {
        orc_fluence(m, leaves + (size_t)b * 2 * m->n_pairs, jaws + (size_t)b * 4, NULL, NULL, NULL, Phimap);
        orc_radiological_depth(g, rho, m, gantry_deg[b], z);
        orc_fan_depth(g, rho, m, gantry_deg[b], zf);
        orc_fan_factor(g, m, zf, z, F);
        orc_project(g, m, Phimap, Phivol);
        orc_apply_fan_factor(g, m, F, Phivol);
        orc_convolve(g, m, W_tab, z, Phivol, Db);
        orc_resample_add(g, m, gantry_deg[b], m->cal * mu[b], Db, dose);
    }
    free(Db); free(Phivol); free(Phimap); free(z); free(zf); free(F);
}
void orc_dose_backward_fan(const orc_grid *g, const orc_model *m, const float *rho, const double *W_tab, int n_cp,
                           const double *leaves, const double *jaws, const double *gantry_deg, const double *mu,
                           const float *gdose, double *d_leaves, double *d_jaws, double *d_mu)
{
    const size_t nb = (size_t)m->beam_nu * g->nz * m->beam_nw, nf = (size_t)m->flu_nu * m->flu_nv;
    const int np = m->n_pairs;
    double *G = malloc(sizeof(double) * nb), *H = malloc(sizeof(double) * nb), *z = malloc(sizeof(double) * m->beam_nw);
    double *Phimap = malloc(sizeof(double) * nf), *gPhimap = malloc(sizeof(double) * nf);
    double *zf = malloc(sizeof(double) * nf * m->beam_nw), *F = malloc(sizeof(double) * nf * m->beam_nw);
    for (int b = 0; b < n_cp; ++b) {
        const double *lv = leaves + (size_t)b * 2 * np, *jw = jaws + (size_t)b * 4;
        orc_fluence(m, lv, jw, NULL, NULL, NULL, Phimap);
        orc_radiological_depth(g, rho, m, gantry_deg[b], z);
        orc_fan_depth(g, rho, m, gantry_deg[b], zf);
        orc_fan_factor(g, m, zf, z, F);
        orc_resample_adjoint(g, m, gantry_deg[b], gdose, G);
        orc_convolve_adjoint(g, m, W_tab, z, G, H);
        orc_apply_fan_factor(g, m, F, H);
        orc_project_adjoint(g, m, H, gPhimap);
        double dot = 0.0;
        for (size_t e = 0; e < nf; ++e) dot += Phimap[e] * gPhimap[e];
        d_mu[b] = m->cal * dot;
        orc_fluence_adjoint(m, lv, jw, gPhimap, d_leaves + (size_t)b * 2 * np, d_jaws + (size_t)b * 4);
        for (int e = 0; e < 2 * np; ++e) d_leaves[(size_t)b * 2 * np + e] *= m->cal * mu[b];
        for (int e = 0; e < 4; ++e) d_jaws[(size_t)b * 4 + e] *= m->cal * mu[b];
    }
    free(G); free(H); free(z); free(Phimap); free(gPhimap); free(zf); free(F);
}

/* ================================================================== collimator rotation */
/* "For non-zero collimator angles, the fluence map is rotated in the beam's eye view about the beam central
 * axis ... applied prior to ray-based projection."  Reading G25: the aperture point (uf, vf) of the collimator
 * frame appears at R(phi_c) (uf, vf) in the beam frame, R the counter-clockwise rotation in the (u, v) plane; the rotated
 * map is the bilinear_0 resampling of the collimator-frame map on the same pixel grid:
 *     Phirot[b][a] = bilinear_0(Phimap; R(-phi_c) (uf_a, vf_b) / (Du, Dv) + centre).                                   */
void orc_rotate_map(const orc_model *m, double coll_deg, const double *Phimap, double *Phirot)
{
    const int nu = m->flu_nu, nv = m->flu_nv;
    const double phi = coll_deg * ORC_PI / 180.0, c = cos(phi), s = sin(phi);
    for (int b = 0; b < nv; ++b)
        for (int a = 0; a < nu; ++a) {
            double u = flu_u(m, a), v = flu_v(m, b);
            double uc = c * u + s * v, vc = -s * u + c * v;                 /* R(-phi_c) (u, v) */
            Phirot[(size_t)b * nu + a] = bilinear0(Phimap, nu, nv, uc / m->flu_du + 0.5 * (nu - 1), vc / m->flu_dv + 0.5 * (nv - 1));
        }
}
/* Transpose of orc_rotate_map, written as the scatter that mirrors it. */
void orc_rotate_map_adjoint(const orc_model *m, double coll_deg, const double *gPhirot, double *gPhimap)
{
    const int nu = m->flu_nu, nv = m->flu_nv;
    const double phi = coll_deg * ORC_PI / 180.0, c = cos(phi), s = sin(phi);
    memset(gPhimap, 0, sizeof(double) * (size_t)nu * nv);
    for (int b = 0; b < nv; ++b)
        for (int a = 0; a < nu; ++a) {
            double u = flu_u(m, a), v = flu_v(m, b);
            double f0 = (c * u + s * v) / m->flu_du + 0.5 * (nu - 1), f1 = (-s * u + c * v) / m->flu_dv + 0.5 * (nv - 1);
            int i0 = (int)floor(f0), i1 = (int)floor(f1);
            double t0 = f0 - i0, t1 = f1 - i1;
            for (int q = 0; q < 4; ++q) {
                int x = i0 + (q & 1), y = i1 + (q >> 1);
                if (x < 0 || x >= nu || y < 0 || y >= nv) continue;
                gPhimap[(size_t)y * nu + x] += ((q & 1) ? t0 : 1.0 - t0) * ((q >> 1) ? t1 : 1.0 - t1) * gPhirot[(size_t)b * nu + a];
            }
        }
}
/* Whole path with per-control-point collimator angles (coll_deg[n_cp]): as orc_dose / orc_dose_backward with the map
 * rotated between the fluence layer and the projection. */
void orc_dose_coll(const orc_grid *g, const orc_model *m, const float *rho, const double *W_tab, int n_cp,
                   const double *leaves, const double *jaws, const double *gantry_deg, const double *coll_deg, const double *mu, double *dose)
{
    const size_t nb = (size_t)m->beam_nu * g->nz * m->beam_nw, np = (size_t)g->nx * g->ny * g->nz, nf = (size_t)m->flu_nu * m->flu_nv;
    double *Db = malloc(sizeof(double) * nb), *Phivol = malloc(sizeof(double) * nb);
    double *Phimap = malloc(sizeof(double) * nf), *Phirot = malloc(sizeof(double) * nf), *z = malloc(sizeof(double) * m->beam_nw);
    memset(dose, 0, sizeof(double) * np);
    for (int b = 0; b < n_cp; ++b) {
        orc_fluence(m, leaves + (size_t)b * 2 * m->n_pairs, jaws + (size_t)b * 4, NULL, NULL, NULL, Phimap);
        orc_rotate_map(m, coll_deg[b], Phimap, Phirot);
        orc_radiological_depth(g, rho, m, gantry_deg[b], z);
        orc_project(g, m, Phirot, Phivol);
        orc_convolve(g, m, W_tab, z, Phivol, Db);
        orc_resample_add(g, m, gantry_deg[b], m->cal * mu[b], Db, dose);
    }
    free(Db); free(Phivol); free(Phimap); free(Phirot); free(z);
}
void orc_dose_backward_coll(const orc_grid *g, const orc_model *m, const float *rho, const double *W_tab, int n_cp,
                            const double *leaves, const double *jaws, const double *gantry_deg, const double *coll_deg, const double *mu,
                            const float *gdose, double *d_leaves, double *d_jaws, double *d_mu)
{
    const size_t nb = (size_t)m->beam_nu * g->nz * m->beam_nw, nf = (size_t)m->flu_nu * m->flu_nv;
    const int np = m->n_pairs;
    double *G = malloc(sizeof(double) * nb), *H = malloc(sizeof(double) * nb), *z = malloc(sizeof(double) * m->beam_nw);
    double *Phimap = malloc(sizeof(double) * nf), *Phirot = malloc(sizeof(double) * nf);
    double *gPhirot = malloc(sizeof(double) * nf), *gPhimap = malloc(sizeof(double) * nf);
    for (int b = 0; b < n_cp; ++b) {
        const double *lv = leaves + (size_t)b * 2 * np, *jw = jaws + (size_t)b * 4;
        orc_fluence(m, lv, jw, NULL, NULL, NULL, Phimap);
        orc_rotate_map(m, coll_deg[b], Phimap, Phirot);
        orc_radiological_depth(g, rho, m, gantry_deg[b], z);
        orc_resample_adjoint(g, m, gantry_deg[b], gdose, G);
        orc_convolve_adjoint(g, m, W_tab, z, G, H);
        orc_project_adjoint(g, m, H, gPhirot);
        double dot = 0.0;
        for (size_t e = 0; e < nf; ++e) dot += Phirot[e] * gPhirot[e];
        d_mu[b] = m->cal * dot;
        orc_rotate_map_adjoint(m, coll_deg[b], gPhirot, gPhimap);
        orc_fluence_adjoint(m, lv, jw, gPhimap, d_leaves + (size_t)b * 2 * np, d_jaws + (size_t)b * 4);
        for (int e = 0; e < 2 * np; ++e) d_leaves[(size_t)b * 2 * np + e] *= m->cal * mu[b];
        for (int e = 0; e < 4; ++e) d_jaws[(size_t)b * 4 + e] *= m->cal * mu[b];
    }
    free(G); free(H); free(z); free(Phimap); free(Phirot); free(gPhirot); free(gPhimap);
}

/* ================================================================== divergent depth AND collimator rotation together */
/* The two optional steps compose in the paper's order ("rotated ... prior to ray-based projection"; reading G24: the
 * depth factor lives at the ray nodes of the beam frame and weights the PROJECTED fluence): fluence -> rotation (G25) -> projection
 * (Eq. 5-6) -> depth factor (G24) -> convolution -> resampling.  No new arithmetic: every step is one of the functions above. */
void orc_dose_fan_coll(const orc_grid *g, const orc_model *m, const float *rho, const double *W_tab, int n_cp,
                       const double *leaves, const double *jaws, const double *gantry_deg, const double *coll_deg, const double *mu, double *dose)
{
    const size_t nb = (size_t)m->beam_nu * g->nz * m->beam_nw, np = (size_t)g->nx * g->ny * g->nz, nf = (size_t)m->flu_nu * m->flu_nv;
    double *Db = malloc(sizeof(double) * nb), *Phivol = malloc(sizeof(double) * nb);
    double *Phimap = malloc(sizeof(double) * nf), *Phirot = malloc(sizeof(double) * nf), *z = malloc(sizeof(double) * m->beam_nw);
    double *zf = malloc(sizeof(double) * nf * m->beam_nw), *F = malloc(sizeof(double) * nf * m->beam_nw);
    memset(dose, 0, sizeof(double) * np);
    for (int b = 0; b < n_cp; ++b) {
        orc_fluence(m, leaves + (size_t)b * 2 * m->n_pairs, jaws + (size_t)b * 4, NULL, NULL, NULL, Phimap);
        orc_rotate_map(m, coll_deg[b], Phimap, Phirot);
        orc_radiological_depth(g, rho, m, gantry_deg[b], z);
        orc_fan_depth(g, rho, m, gantry_deg[b], zf);
        orc_fan_factor(g, m, zf, z, F);
        orc_project(g, m, Phirot, Phivol);
        orc_apply_fan_factor(g, m, F, Phivol);
        orc_convolve(g, m, W_tab, z, Phivol, Db);
        orc_resample_add(g, m, gantry_deg[b], m->cal * mu[b], Db, dose);
    }
    free(Db); free(Phivol); free(Phimap); free(Phirot); free(z); free(zf); free(F);
}
void orc_dose_backward_fan_coll(const orc_grid *g, const orc_model *m, const float *rho, const double *W_tab, int n_cp,
                                const double *leaves, const double *jaws, const double *gantry_deg, const double *coll_deg, const double *mu,
                                const float *gdose, double *d_leaves, double *d_jaws, double *d_mu)
{
    const size_t nb = (size_t)m->beam_nu * g->nz * m->beam_nw, nf = (size_t)m->flu_nu * m->flu_nv;
    const int np = m->n_pairs;
    double *G = malloc(sizeof(double) * nb), *H = malloc(sizeof(double) * nb), *z = malloc(sizeof(double) * m->beam_nw);
    double *Phimap = malloc(sizeof(double) * nf), *Phirot = malloc(sizeof(double) * nf);
    double *gPhirot = malloc(sizeof(double) * nf), *gPhimap = malloc(sizeof(double) * nf);
    double *zf = malloc(sizeof(double) * nf * m->beam_nw), *F = malloc(sizeof(double) * nf * m->beam_nw);
    for (int b = 0; b < n_cp; ++b) {
        const double *lv = leaves + (size_t)b * 2 * np, *jw = jaws + (size_t)b * 4;
        orc_fluence(m, lv, jw, NULL, NULL, NULL, Phimap);
        orc_rotate_map(m, coll_deg[b], Phimap, Phirot);
        orc_radiological_depth(g, rho, m, gantry_deg[b], z);
        orc_fan_depth(g, rho, m, gantry_deg[b], zf);
        orc_fan_factor(g, m, zf, z, F);
        orc_resample_adjoint(g, m, gantry_deg[b], gdose, G);
        orc_convolve_adjoint(g, m, W_tab, z, G, H);
        orc_apply_fan_factor(g, m, F, H);
        orc_project_adjoint(g, m, H, gPhirot);
        double dot = 0.0;
        for (size_t e = 0; e < nf; ++e) dot += Phirot[e] * gPhirot[e];
        d_mu[b] = m->cal * dot;
        orc_rotate_map_adjoint(m, coll_deg[b], gPhirot, gPhimap);
        orc_fluence_adjoint(m, lv, jw, gPhimap, d_leaves + (size_t)b * 2 * np, d_jaws + (size_t)b * 4);
        for (int e = 0; e < 2 * np; ++e) d_leaves[(size_t)b * 2 * np + e] *= m->cal * mu[b];
        for (int e = 0; e < 4; ++e) d_jaws[(size_t)b * 4 + e] *= m->cal * mu[b];
    }
    free(G); free(H); free(z); free(Phimap); free(Phirot); free(gPhirot); free(gPhimap); free(zf); free(F);
}

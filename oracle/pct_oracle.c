/*
 * pct_oracle.c -- plain, slow CPU ORACLE for the pCT hot path.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may build, load or call it.
 * It shares no code, header, table generator or constant generator with the CUDA
 * path under paper_1707_05014_b200/csrc/ and neither includes the other.
 *
 * What it computes (citations: PAPER.md = /root/reference/PAPER.md of arxiv 1707.05014;
 * DESIGN.md section "Readings" R1..R23 and section "The rule" = the written fp32 rule):
 *
 *   history (entry/exit position + direction at the tracker planes, WEPL)  PAPER.md:42 (sec. 2)
 *     -> straight rays to the object hull                                   DESIGN.md R6,R7
 *     -> most-likely path (2x2 scattering-matrix maximum likelihood)        PAPER.md:42, R2-R5
 *     -> voxel walk: sparse row a_i of A (voxel index, chord length)        PAPER.md:44, R9-R11
 *     -> block-iterative diagonally relaxed projections (DROP) on Ax=b      PAPER.md:44-50, Fig. 1, R12-R18
 *
 * Two tiers:
 *   T64  everything in fp64 from the definitions: matrix form of the MLP with explicit
 *        2x2 inverses, exact integrals of the scattering polynomial, libm log.
 *   T32  a scalar mirror of the fp32 rule: the voxel index of a segment is decided by
 *        floor() of an fp32 midpoint, so both sides take that decision in the same
 *        precision and op order.  The DROP loop takes its rows from T32 (lengths
 *        promoted to double) and accumulates everything (dot, norm, residual, Delta, x)
 *        in fp64.
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): cubic-spline closed form of the MLP,
 * brute-force likelihood maximisation, quadrature of the scattering integrals,
 * straight-line limit / shear equivariance, exact endpoints, chord-length sum,
 * log-factor cancellation at mid-depth, kinematics of the constants, the worked
 * example of SURVEY.md Appendix A, Kaczmarz single-row identity, hit-count identities,
 * block structure, convergence to a dense least-squares solve on a 6x6x4 grid.
 * Unpinned: absolute reconstruction accuracy against a real phantom scan
 * (Table 2) -- "parity unpinned", the scan data do not exist here.
 *
 * Build: gcc -O2 -ffp-contract=off -fno-fast-math [-mfma] -fopenmp -shared -fPIC
 * (-ffp-contract=off is REQUIRED: the fp32 rule names every fused multiply-add itself).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* ------------------------------------------------------------------------------------------
 * Constants (step 0).  Build constants of the cited formalism, not in
 * PAPER.md (reading R3): 1/(beta^2 p^2) of 200 MeV protons in water as a 5th-degree polynomial
 * of depth, radiation length of water, Highland log coefficient.
 * ---------------------------------------------------------------------------------------- */
#define ORC_X0_MM 361.0
#define ORC_LOGC 0.038
#define ORC_EPS (1.0 / 1024.0) /* 2^-10 mm */
#define ORC_SCALE 8192.0       /* common scale 2^13 of Sigma1 and Sigma2; cancels in the MLP */

/* a_k in c^2/MeV^2 per cm^k (depth in cm) */
static const double ORC_A_CM[6] = {7.457e-6, 4.548e-7, -5.777e-8, 1.301e-8, -9.228e-10, 2.687e-11};

/* fp32 polynomial coefficients per mm^k times 2^13, the rule's constants A0..A5 (hex floats) */
static const float RA0 = 0x1.f46e48p-5f;
static const float RA1 = 0x1.86ab94p-12f;
static const float RA2 = -0x1.3d980cp-18f;
static const float RA3 = 0x1.c9bfaap-24f;
static const float RA4 = -0x1.9f9798p-31f;
static const float RA5 = 0x1.35ca3ep-39f;

/* rule_log constants: ln2, and P(t) ~ ln(1+t)/t on [sqrt(1/2)-1, sqrt(2)-1], degree 5 */
static const float RLN2 = 0x1.62e43p-1f;
static const float RLP0 = 0x1.00004ep+0f;
static const float RLP1 = -0x1.ffe6bcp-2f;
static const float RLP2 = 0x1.548ca6p-2f;
static const float RLP3 = -0x1.0412e4p-2f;
static const float RLP4 = 0x1.c3ffeep-3f;
static const float RLP5 = -0x1.25a60ep-3f;
static const float RINVX0 = 0x1.6b1490p-9f; /* fp32(1/361) */
static const float RLOGC = 0x1.374bc6p-5f;  /* fp32(0.038) */
static const float REPS = 0x1p-10f;

typedef struct {
    int nx, ny, nz;
    float h;     /* voxel edge, mm */
    float u_in;  /* depth of the entry tracker plane in the beam frame, mm (<= -R_h) */
    float u_out; /* depth of the exit tracker plane, mm (>= +R_h) */
} orc_geom;

/* mm-based fp64 polynomial coefficient a_j * 10^-j (unscaled) */
static double a_mm(const double *a_cm, int j) {
    double v = a_cm[j];
    for (int i = 0; i < j; ++i) v *= 0.1;
    return v;
}

/* ==========================================================================================
 * T64: definitions in fp64
 * ======================================================================================== */

/* Integrals of the scattering polynomial f(s) = sum_j a_j s^j over [lo, hi]:
 *   n=2: A = int (ref - s)^2 f(s) ds,  n=1: B = int (ref - s) f(s) ds,  n=0: C = int f(s) ds
 * by 8-point Gauss-Legendre quadrature, which is exact (up to rounding) for the degree <= 7
 * integrands here and has no cancellation (f > 0 on the supported depth range). */
static double poly_moment(const double *a, double lo, double hi, double ref, int n) {
    static const double gx[8] = {-0.96028985649753618, -0.79666647741362673, -0.52553240991632899,
                                 -0.18343464249564978, 0.18343464249564978,  0.52553240991632899,
                                 0.79666647741362673,  0.96028985649753618};
    static const double gw[8] = {0.10122853629037706, 0.22238103445337443, 0.31370664587788688,
                                 0.36268378337836166, 0.36268378337836166, 0.31370664587788688,
                                 0.22238103445337443, 0.10122853629037706};
    const double mid = 0.5 * (lo + hi), half = 0.5 * (hi - lo);
    double total = 0.0;
    for (int q = 0; q < 8; ++q) {
        const double s = mid + half * gx[q];
        double f = 0.0;
        for (int j = 5; j >= 0; --j) f = f * s + a[j];
        double wgt = 1.0;
        for (int m = 0; m < n; ++m) wgt *= (ref - s);
        total += gw[q] * wgt * f;
    }
    return total * half;
}

static double highland_K(double d) {
    double g = 1.0 + ORC_LOGC * log(d / ORC_X0_MM);
    return g * g;
}

static void inv2(const double m[4], double out[4]) {
    double det = m[0] * m[3] - m[1] * m[2];
    out[0] = m[3] / det;
    out[1] = -m[1] / det;
    out[2] = -m[2] / det;
    out[3] = m[0] / det;
}
static void mul22(const double a[4], const double b[4], double c[4]) {
    c[0] = a[0] * b[0] + a[1] * b[2];
    c[1] = a[0] * b[1] + a[1] * b[3];
    c[2] = a[2] * b[0] + a[3] * b[2];
    c[3] = a[2] * b[1] + a[3] * b[3];
}
static void mul21(const double a[4], const double v[2], double o[2]) {
    o[0] = a[0] * v[0] + a[1] * v[1];
    o[1] = a[2] * v[0] + a[3] * v[1];
}

/* Matrix-form maximum-likelihood path in one plane (R2, the formalism of the
 * Schulte 2008 citation at PAPER.md:42):
 *   y1 = (S1^-1 + R1^T S2^-1 R1)^-1 (S1^-1 R0 y0 + R1^T S2^-1 y2),  y = (t, theta)^T
 *   R0 = [[1,s1],[0,1]], R1 = [[1,L-s1],[0,1]]
 *   S1 = K(s1) [[A1,B1],[B1,C1]] over [0,s1] referenced to s1, S2 = K(L-s1)[[A2,B2],[B2,C2]]
 *   over [s1,L] referenced to L.
 * a_mm6: polynomial coefficients per mm^j (NULL = the build constants); use_log: 0 => K == 1.
 * Returns 0, or -1 if s1 is not strictly inside (0, L). */
int orc_mlp_matrix_f64(double s1, double L, const double y0[2], const double y2[2],
                       const double *a_mm6, int use_log, double y1[2]) {
    double a[6];
    if (!(s1 > 0.0) || !(s1 < L)) return -1;
    for (int j = 0; j < 6; ++j) a[j] = a_mm6 ? a_mm6[j] : a_mm(ORC_A_CM, j);
    double d = L - s1;
    double k1 = use_log ? highland_K(s1) : 1.0;
    double k2 = use_log ? highland_K(d) : 1.0;
    double S1[4] = {k1 * poly_moment(a, 0.0, s1, s1, 2), k1 * poly_moment(a, 0.0, s1, s1, 1),
                    k1 * poly_moment(a, 0.0, s1, s1, 1), k1 * poly_moment(a, 0.0, s1, s1, 0)};
    double S2[4] = {k2 * poly_moment(a, s1, L, L, 2), k2 * poly_moment(a, s1, L, L, 1),
                    k2 * poly_moment(a, s1, L, L, 1), k2 * poly_moment(a, s1, L, L, 0)};
    double R0[4] = {1.0, s1, 0.0, 1.0}, R1[4] = {1.0, d, 0.0, 1.0}, R1T[4] = {1.0, 0.0, d, 1.0};
    double S1i[4], S2i[4], T1[4], T2[4], M[4], Mi[4], v1[2], v2[2], w[2], rhs[2];
    inv2(S1, S1i);
    inv2(S2, S2i);
    mul22(R1T, S2i, T1);  /* R1^T S2^-1       */
    mul22(T1, R1, T2);    /* R1^T S2^-1 R1    */
    for (int i = 0; i < 4; ++i) M[i] = S1i[i] + T2[i];
    mul21(R0, y0, w);     /* R0 y0            */
    mul21(S1i, w, v1);    /* S1^-1 R0 y0      */
    mul21(T1, y2, v2);    /* R1^T S2^-1 y2    */
    rhs[0] = v1[0] + v2[0];
    rhs[1] = v1[1] + v2[1];
    inv2(M, Mi);
    mul21(Mi, rhs, y1);
    return 0;
}

/* The likelihood exponent whose minimum over y1 defines the MLP (used by a brute-force pin):
 * chi2(y1) = (y1 - R0 y0)^T S1^-1 (y1 - R0 y0) + (y2 - R1 y1)^T S2^-1 (y2 - R1 y1). */
double orc_mlp_chi2_f64(double s1, double L, const double y0[2], const double y2[2],
                        const double y1[2], int use_log) {
    double a[6];
    for (int j = 0; j < 6; ++j) a[j] = a_mm(ORC_A_CM, j);
    double d = L - s1;
    double k1 = use_log ? highland_K(s1) : 1.0, k2 = use_log ? highland_K(d) : 1.0;
    double S1[4] = {k1 * poly_moment(a, 0.0, s1, s1, 2), k1 * poly_moment(a, 0.0, s1, s1, 1),
                    k1 * poly_moment(a, 0.0, s1, s1, 1), k1 * poly_moment(a, 0.0, s1, s1, 0)};
    double S2[4] = {k2 * poly_moment(a, s1, L, L, 2), k2 * poly_moment(a, s1, L, L, 1),
                    k2 * poly_moment(a, s1, L, L, 1), k2 * poly_moment(a, s1, L, L, 0)};
    double S1i[4], S2i[4], e1[2], e2[2], t[2];
    inv2(S1, S1i);
    inv2(S2, S2i);
    e1[0] = y1[0] - (y0[0] + s1 * y0[1]);
    e1[1] = y1[1] - y0[1];
    e2[0] = y2[0] - (y1[0] + d * y1[1]);
    e2[1] = y2[1] - y1[1];
    mul21(S1i, e1, t);
    double c = e1[0] * t[0] + e1[1] * t[1];
    mul21(S2i, e2, t);
    return c + e2[0] * t[0] + e2[1] * t[1];
}

/* scattering polynomial and its integrals, exported for the quadrature / kinematics pins.
 * f in c^2/MeV^2 (unscaled), s in mm */
double orc_scatter_f(double s_mm) {
    double v = 0.0;
    for (int j = 5; j >= 0; --j) v = v * s_mm + a_mm(ORC_A_CM, j);
    return v;
}
void orc_sigma_f64(double s1, double L, double S1[3], double S2[3]) {
    double a[6];
    for (int j = 0; j < 6; ++j) a[j] = a_mm(ORC_A_CM, j);
    for (int n = 0; n < 3; ++n) {
        S1[2 - n] = poly_moment(a, 0.0, s1, s1, n); /* S[0]=A (n=2), S[1]=B, S[2]=C */
        S2[2 - n] = poly_moment(a, s1, L, L, n);
    }
}

typedef struct {
    float t_in, v_in, t_out, v_out;       /* positions at the tracker planes, mm */
    float tht_in, thv_in, tht_out, thv_out; /* slopes dt/du, dv/du */
    float cs, sn;                         /* cos, sin of the projection angle (caller's fp32 table) */
} orc_hist;

/* T64 hull + MLP nodes in the object frame.  nodes: (K+2) x 3 doubles.  Returns the number of
 * nodes (K+2), 0 if the history is skipped, or -needed if max_nodes is too small.
 * hullout (optional, 7 doubles): u0,t0,v0,u2,t2,v2,L. */
/* Path model (R30).  0: the most-likely path of the scattering-matrix
 * formalism (the graded path).  1: the CUBIC SPLINE through the hull entry and exit points with the measured
 * directions -- what the MLP becomes for a constant scattering power (pin P1) -- as a cheap mode:
 *     t(s) = t0 + sigma s + c0 alpha0 + c2 alpha2,  c0 = L tau (1 - tau)^2,  c2 = -L tau^2 (1 - tau),  tau = s / L
 * in the chord frame (alpha = direction - chord slope sigma); same for v. */
static int g_path_model = 0;
void orc_set_path_model(int m) { g_path_model = m == 1 ? 1 : 0; }
int orc_get_path_model(void) { return g_path_model; }

/* Depth step of the path (R33).  1: one voxel edge h (R9, the graded path).
 * 2: the HALF-VOXEL step h/2 -- nodes at depth k h/2, K = floor((L - eps) / (h/2)) capped at 2 min(nx, ny), the
 * Sigma1^-1 table at s = k h/2; everything else (hull, coefficients, voxel rule, merge, DROP) unchanged. */
static int g_substeps = 1;
void orc_set_substeps(int n) { g_substeps = n == 2 ? 2 : 1; }
int orc_get_substeps(void) { return g_substeps; }
static float r32_step(const orc_geom *g) { return g_substeps == 2 ? 0.5f * g->h : g->h; }
static int orc_kmax(const orc_geom *g) { return g_substeps * (g->nx < g->ny ? g->nx : g->ny); }
float orc_step(const orc_geom *g) { return r32_step(g); }

static double spline_f64(double s1, double L, const double y0[2], const double y2[2]) {
    const double sigma = (y2[0] - y0[0]) / L, a0 = y0[1] - sigma, a2 = y2[1] - sigma, tau = s1 / L;
    return y0[0] + sigma * s1 + L * tau * (1.0 - tau) * (1.0 - tau) * a0 - L * tau * tau * (1.0 - tau) * a2;
}

int orc_path_f64(const orc_geom *g, const orc_hist *hh, int max_nodes, double *nodes, double *hullout) {
    double h = (double)g->h;
    int nmin = g->nx < g->ny ? g->nx : g->ny;
    double R = 0.5 * h * nmin, zmax = 0.5 * h * g->nz;
    double u_in = g->u_in, u_out = g->u_out;
    double th0 = hh->tht_in, th2 = hh->tht_out, ph0 = hh->thv_in, ph2 = hh->thv_out;
    /* step 1: straight rays in air onto the hull cylinder t^2 + u^2 = R^2 (R6, R7) */
    double c0 = hh->t_in - th0 * u_in, q0 = 1.0 + th0 * th0;
    double disc0 = R * R * q0 - c0 * c0;
    double c2 = hh->t_out - th2 * u_out, q2 = 1.0 + th2 * th2;
    double disc2 = R * R * q2 - c2 * c2;
    if (!(disc0 > 0.0) || !(disc2 > 0.0)) return 0;
    double u0 = (-th0 * c0 - sqrt(disc0)) / q0; /* first crossing of the entry ray  */
    double u2 = (-th2 * c2 + sqrt(disc2)) / q2; /* last crossing of the exit ray    */
    double t0 = c0 + th0 * u0, v0 = hh->v_in + ph0 * (u0 - u_in);
    double t2 = c2 + th2 * u2, v2 = hh->v_out + ph2 * (u2 - u_out);
    double L = u2 - u0;
    if (!(L > ORC_EPS) || fabs(v0) > zmax || fabs(v2) > zmax) return 0;
    if (hullout) {
        hullout[0] = u0; hullout[1] = t0; hullout[2] = v0;
        hullout[3] = u2; hullout[4] = t2; hullout[5] = v2; hullout[6] = L;
    }
    const double step = h / (double)g_substeps;
    int K = (int)floor((L - ORC_EPS) / step);
    if (K + 2 > max_nodes) return -(K + 2);
    double cs = hh->cs, sn = hh->sn;
    for (int k = 0; k <= K + 1; ++k) {
        double t, u, v;
        if (k == 0) { t = t0; u = u0; v = v0; }
        else if (k == K + 1) { t = t2; u = u2; v = v2; }
        else {
            double s1 = k * step;
            double yt0[2] = {t0, th0}, yt2[2] = {t2, th2}, yv0[2] = {v0, ph0}, yv2[2] = {v2, ph2};
            double y[2];
            if (g_path_model == 1) {
                t = spline_f64(s1, L, yt0, yt2);
                v = spline_f64(s1, L, yv0, yv2);
            } else {
                orc_mlp_matrix_f64(s1, L, yt0, yt2, NULL, 1, y);
                t = y[0];
                orc_mlp_matrix_f64(s1, L, yv0, yv2, NULL, 1, y);
                v = y[0];
            }
            u = u0 + s1;
        }
        nodes[3 * k + 0] = t * cs - u * sn; /* rotation about z by the projection angle (R8) */
        nodes[3 * k + 1] = t * sn + u * cs;
        nodes[3 * k + 2] = v;
    }
    return K + 2;
}

/* ==========================================================================================
 * Sigma1^-1 table (step T): fp64 closed forms rounded once to fp32.
 * Entry k (1..kmax) at depth s = k*h:  P = (K(s) [[A1,B1],[B1,C1]] * 2^13)^-1 = (p11,p12,p22).
 * ======================================================================================== */
int orc_sigma1_table(float h32, int kmax, float *p11, float *p12, float *p22) {
    double h = (double)h32;
    for (int k = 0; k <= kmax; ++k) {
        if (k == 0) { p11[0] = p12[0] = p22[0] = 0.0f; continue; }
        double s = (double)k * h;
        double A = 0.0, B = 0.0, C = 0.0, sp = s; /* sp = s^(j+1) */
        for (int j = 0; j < 6; ++j) {
            double aj = a_mm(ORC_A_CM, j) * ORC_SCALE;
            C += aj * sp / (double)(j + 1);
            B += aj * sp * s / (double)((j + 1) * (j + 2));
            A += 2.0 * aj * sp * s * s / (double)((j + 1) * (j + 2) * (j + 3));
            sp *= s;
        }
        double W = highland_K(s) * (A * C - B * B);
        p11[k] = (float)(C / W);
        p12[k] = (float)(-B / W);
        p22[k] = (float)(A / W);
    }
    return 0;
}

/* ==========================================================================================
 * T32: scalar mirror of the fp32 rule.  Every operation below is one
 * IEEE fp32 operation; fmaf is used exactly where the rule writes fma(.,.,.).
 * ======================================================================================== */

/* rule_log(x), x a positive normal float: ln x = e ln2 + t P(t), x = m 2^e, m in [sqrt(.5), sqrt 2) */
static float rule_log(float x) {
    int32_t bits;
    memcpy(&bits, &x, 4);
    int32_t e = (bits - 0x3f3504f3) >> 23; /* arithmetic shift */
    int32_t mb = bits - (int32_t)((uint32_t)e << 23);
    float m;
    memcpy(&m, &mb, 4);
    float t = m - 1.0f;
    float p = RLP5;
    p = fmaf(p, t, RLP4);
    p = fmaf(p, t, RLP3);
    p = fmaf(p, t, RLP2);
    p = fmaf(p, t, RLP1);
    p = fmaf(p, t, RLP0);
    return fmaf((float)e, RLN2, t * p);
}
float orc_rule_log(float x) { return rule_log(x); }

typedef struct {
    /* hull */
    float u0, t0, v0, u2, t2, v2, L;
    /* chord frame */
    float sig_t, sig_v, al0, al2, be0, be2;
    /* integrated Taylor-shift coefficients of f(L - w) */
    float qc[6], qb[6], qa[6];
    int K;
} r32_state;

/* c + cl = t_pl - theta*u_pl to about twice fp32 precision: p + pe = theta*u_pl exactly (fma),
 * c + e = t_pl - p exactly (two-sum), cl = e - pe. */
static void r32_ray_offset(float t_pl, float theta, float u_pl, float *c_out, float *cl_out) {
    const float p = theta * u_pl;
    const float pe = fmaf(theta, u_pl, -p);
    const float c = t_pl - p;
    const float bb = c - t_pl;
    const float e = (t_pl - (c - bb)) + (-p - bb);
    *c_out = c;
    *cl_out = e - pe;
}

/* hull + per-history set-up.  Returns 1 if the history has a path, 0 if skipped (R7). */
static int r32_setup(const orc_geom *g, const orc_hist *hh, r32_state *st) {
    const float h = g->h;
    const float inv_h = 1.0f / h;
    const int nmin = g->nx < g->ny ? g->nx : g->ny;
    const float R = (0.5f * h) * (float)nmin;
    const float R2 = R * R;
    const float zmax = (0.5f * (float)g->nz) * h;
    /* step 1: ray t = c + theta*u with c = t_pl - theta*u_pl carried as c + cl (product and sum
     * errors recovered exactly), discriminant R^2(1+theta^2) - c^2 = (R-c)(R+c) + R^2 theta^2:
     * no cancellation of rounded squares, so grazing rays keep their hull points to ~1e-5 mm */
    float c_in, cl_in, c_out, cl_out;
    r32_ray_offset(hh->t_in, hh->tht_in, g->u_in, &c_in, &cl_in);
    r32_ray_offset(hh->t_out, hh->tht_out, g->u_out, &c_out, &cl_out);
    const float q_in = fmaf(hh->tht_in, hh->tht_in, 1.0f);
    const float q_out = fmaf(hh->tht_out, hh->tht_out, 1.0f);
    const float disc_in = fmaf((R - c_in) - cl_in, (R + c_in) + cl_in, R2 * (hh->tht_in * hh->tht_in));
    const float disc_out = fmaf((R - c_out) - cl_out, (R + c_out) + cl_out, R2 * (hh->tht_out * hh->tht_out));
    if (!(disc_in > 0.0f) || !(disc_out > 0.0f)) return 0;
    const float u0 = fmaf(-hh->tht_in, c_in, -sqrtf(disc_in)) / q_in;
    const float u2 = fmaf(-hh->tht_out, c_out, sqrtf(disc_out)) / q_out;
    const float t0 = fmaf(hh->tht_in, u0, c_in);
    const float v0 = fmaf(hh->thv_in, u0 - g->u_in, hh->v_in);
    const float t2 = fmaf(hh->tht_out, u2, c_out);
    const float v2 = fmaf(hh->thv_out, u2 - g->u_out, hh->v_out);
    const float L = u2 - u0;
    if (!(L > REPS) || !(fabsf(v0) <= zmax) || !(fabsf(v2) <= zmax)) return 0;
    st->u0 = u0; st->t0 = t0; st->v0 = v0; st->u2 = u2; st->t2 = t2; st->v2 = v2; st->L = L;
    /* step 2 */
    const float invL = 1.0f / L;
    st->sig_t = (t2 - t0) * invL;
    st->sig_v = (v2 - v0) * invL;
    st->al0 = hh->tht_in - st->sig_t;
    st->al2 = hh->tht_out - st->sig_t;
    st->be0 = hh->thv_in - st->sig_v;
    st->be2 = hh->thv_out - st->sig_v;
    /* Taylor shift f(L - w) = sum_j q_j w^j, q_j = (-1)^j sum_{m>=j} binom(m,j) a_m L^(m-j) */
    float q[6];
    q[0] = fmaf(fmaf(fmaf(fmaf(fmaf(RA5, L, RA4), L, RA3), L, RA2), L, RA1), L, RA0);
    q[1] = -fmaf(fmaf(fmaf(fmaf(5.0f * RA5, L, 4.0f * RA4), L, 3.0f * RA3), L, 2.0f * RA2), L, RA1);
    q[2] = fmaf(fmaf(fmaf(10.0f * RA5, L, 6.0f * RA4), L, 3.0f * RA3), L, RA2);
    q[3] = -fmaf(fmaf(10.0f * RA5, L, 4.0f * RA4), L, RA3);
    q[4] = fmaf(5.0f * RA5, L, RA4);
    q[5] = -RA5;
    for (int j = 0; j < 6; ++j) {
        st->qc[j] = q[j] * (1.0f / (float)(j + 1));
        st->qb[j] = q[j] * (1.0f / (float)(j + 2));
        st->qa[j] = q[j] * (1.0f / (float)(j + 3));
    }
    /* step 4 node count */
    const float inv_step = 1.0f / r32_step(g);
    int K = (int)floorf((L - REPS) * inv_step);
    if (K > orc_kmax(g)) K = orc_kmax(g);
    st->K = K;
    return 1;
}

/* step 3: MLP coefficients (c0, c2) at node k (1..K); tab = Sigma1^-1 table */
static void r32_coef(const r32_state *st, float h, int k, const float *p11t, const float *p12t,
                     const float *p22t, float *s1_out, float *c0_out, float *c2_out) {
    const float s1 = (float)k * h;
    if (g_path_model == 1) { /* spline rule (R30): five fp32 operations after tau = s1 * (1/L) */
        const float invL = 1.0f / st->L;
        const float tau = s1 * invL;
        const float om = 1.0f - tau;
        const float a = tau * om;
        *s1_out = s1;
        *c0_out = (a * om) * st->L;
        *c2_out = -((a * tau) * st->L);
        return;
    }
    const float d = st->L - s1;
    const float p11 = p11t[k], p12 = p12t[k], p22 = p22t[k];
    const float e1 = fmaf(p11, s1, p12);
    const float f1 = fmaf(p12, s1, p22);
    const float d2 = d * d, d3 = d2 * d;
    float hc = st->qc[5], hb = st->qb[5], ha = st->qa[5];
    for (int j = 4; j >= 0; --j) {
        hc = fmaf(hc, d, st->qc[j]);
        hb = fmaf(hb, d, st->qb[j]);
        ha = fmaf(ha, d, st->qa[j]);
    }
    const float C2 = hc * d, B2 = hb * d2, A2 = ha * d3;
    const float det2 = fmaf(A2, C2, -(B2 * B2));
    const float lg = rule_log(d * RINVX0);
    const float kk = fmaf(RLOGC, lg, 1.0f);
    const float w1 = (kk * kk) * det2;
    const float n12 = fmaf(C2, d, -B2);
    const float gg = fmaf(-B2, d, A2);
    const float n22 = fmaf(d, n12, gg);
    const float m11 = fmaf(w1, p11, C2);
    const float m12 = fmaf(w1, p12, n12);
    const float m22 = fmaf(w1, p22, n22);
    const float det = fmaf(m11, m22, -(m12 * m12));
    const float rdet = 1.0f / det;
    const float num0 = w1 * fmaf(m22, e1, -(m12 * f1));
    const float num2 = -fmaf(m22, B2, m12 * gg);
    *s1_out = s1;
    *c0_out = num0 * rdet;
    *c2_out = num2 * rdet;
}

static void r32_node(const orc_geom *g, const orc_hist *hh, const r32_state *st, int k,
                     const float *p11t, const float *p12t, const float *p22t, float xyz[3]) {
    float t, u, v;
    if (k == 0) { t = st->t0; u = st->u0; v = st->v0; }
    else if (k == st->K + 1) { t = st->t2; u = st->u2; v = st->v2; }
    else {
        float s1, c0, c2;
        r32_coef(st, r32_step(g), k, p11t, p12t, p22t, &s1, &c0, &c2);
        t = fmaf(c2, st->al2, fmaf(c0, st->al0, fmaf(st->sig_t, s1, st->t0)));
        v = fmaf(c2, st->be2, fmaf(c0, st->be0, fmaf(st->sig_v, s1, st->v0)));
        u = st->u0 + s1;
    }
    xyz[0] = fmaf(t, hh->cs, -(u * hh->sn));
    xyz[1] = fmaf(t, hh->sn, u * hh->cs);
    xyz[2] = v;
}

/* One history through the fp32 rule.
 *   seg_idx/seg_len  (optional) raw segments k = 0..K: linear voxel index (or -1 if dropped) and length
 *   row_idx/row_len  merged row: consecutive (in k) equal indices merged, dropped segments removed
 *                    and breaking a run (R10)
 *   nodes            (optional) (K+2) x 3 fp32 object-frame node positions
 *   coefs            (optional) (K+2) x 2 fp32 MLP coefficients c0, c2 (0 for the end nodes)
 * Returns nnz of the merged row (0 for a skipped history), or -needed if max_seg < K+1.
 * *nseg_out = K+1 (0 if skipped). */
/* ==========================================================================================
 * Walk mode (R34).  0: the midpoint rule of R10 (a segment's length goes to the
 * voxel of its midpoint), the graded path.  1: EXACT traversal of the polyline: every segment A -> B is cut at
 * the voxel faces it crosses and every piece goes to the voxel it lies in, so that the row is the list of the
 * polyline's chord lengths.  fp32, this operation order (it decides voxel indices):
 *     gA = fma(A, 1/h, n/2), gB likewise, d = gB - gA                       (grid coordinates, per axis)
 *     for axis x, y, z: if floor(gA) != floor(gB): for every integer p, min + 1 <= p <= max of the two floors,
 *         ascending: t = (p - gA) / d, clamped to [0, 1]                    (at most ORC_MAX_CUTS cuts in all)
 *     cuts sorted ascending; consecutive cuts t0 < t1 (0 and 1 included) give a piece of length (t1 - t0) * len
 *     in the voxel floor(fma(0.5 (t0 + t1), d, gA)); pieces of zero length are dropped
 * The row merges consecutive equal voxels as before (a piece outside the grid breaks a run).
 * ======================================================================================== */
#define ORC_MAX_CUTS 24
static int g_walk_mode = 0;
void orc_set_walk_mode(int m) { g_walk_mode = m == 1 ? 1 : 0; }
int orc_get_walk_mode(void) { return g_walk_mode; }
int orc_row_capacity(const orc_geom *g) { return g_walk_mode == 1 ? 8 * (orc_kmax(g) + 2) : orc_kmax(g) + 2; }

static int32_t r32_voxel(const orc_geom *g, float gx, float gy, float gz) {
    const float fx = floorf(gx), fy = floorf(gy), fz = floorf(gz);
    if (fx >= 0.0f && fx < (float)g->nx && fy >= 0.0f && fy < (float)g->ny && fz >= 0.0f && fz < (float)g->nz)
        return (int32_t)fx + g->nx * ((int32_t)fy + g->ny * (int32_t)fz);
    return -1;
}

static int r32_pieces(const orc_geom *g, const float A[3], const float B[3], float len, int32_t *vox, float *plen) {
    const float inv_h = 1.0f / g->h;
    const float half[3] = {0.5f * (float)g->nx, 0.5f * (float)g->ny, 0.5f * (float)g->nz};
    float ga[3], d[3], ts[ORC_MAX_CUTS];
    int nt = 0;
    for (int c = 0; c < 3; ++c) {
        ga[c] = fmaf(A[c], inv_h, half[c]);
        const float gb = fmaf(B[c], inv_h, half[c]);
        d[c] = gb - ga[c];
        const float fa = floorf(ga[c]), fb = floorf(gb);
        if (fa != fb) {
            const float lo = fa < fb ? fa : fb, hi = fa < fb ? fb : fa;
            for (float p = lo + 1.0f; p <= hi && nt < ORC_MAX_CUTS; p += 1.0f) {
                float t = (p - ga[c]) / d[c];
                t = t < 0.0f ? 0.0f : (t > 1.0f ? 1.0f : t);
                ts[nt++] = t;
            }
        }
    }
    for (int i = 1; i < nt; ++i) { /* insertion sort, ascending */
        const float v = ts[i];
        int j = i - 1;
        while (j >= 0 && ts[j] > v) { ts[j + 1] = ts[j]; --j; }
        ts[j + 1] = v;
    }
    int np = 0;
    float t0 = 0.0f;
    for (int j = 0; j <= nt; ++j) {
        const float t1 = j < nt ? ts[j] : 1.0f;
        if (t1 > t0) {
            const float tm = 0.5f * (t0 + t1);
            vox[np] = r32_voxel(g, fmaf(tm, d[0], ga[0]), fmaf(tm, d[1], ga[1]), fmaf(tm, d[2], ga[2]));
            plen[np] = (t1 - t0) * len;
            ++np;
            t0 = t1;
        }
    }
    return np;
}

/* number of nodes K + 2 of the fp32 path of a history (0: skipped) */
int orc_node_count(const orc_geom *g, const orc_hist *hh) {
    r32_state st;
    return r32_setup(g, hh, &st) ? st.K + 2 : 0;
}

int orc_row_f32(const orc_geom *g, const orc_hist *hh, const float *p11t, const float *p12t,
                const float *p22t, int max_seg, int32_t *row_idx, float *row_len, int32_t *seg_idx,
                float *seg_len, float *nodes, float *coefs, int *nseg_out) {
    r32_state st;
    if (nseg_out) *nseg_out = 0;
    if (!r32_setup(g, hh, &st)) return 0;
    const int K = st.K;
    if (K + 1 > max_seg) return -(K + 1);
    const float inv_h = 1.0f / g->h;
    const float hx = 0.5f * (float)g->nx, hy = 0.5f * (float)g->ny, hz = 0.5f * (float)g->nz;
    float prev[3], cur[3];
    int nnz = 0, ns = 0; /* ns: items (segments, or pieces in the exact mode) emitted so far */
    int32_t last = -1;   /* voxel of the previous item (-1: none or dropped) */
    r32_node(g, hh, &st, 0, p11t, p12t, p22t, prev);
    if (nodes) memcpy(nodes, prev, 12);
    if (coefs) { coefs[0] = 0.0f; coefs[1] = 0.0f; }
    for (int k = 0; k <= K; ++k) {
        r32_node(g, hh, &st, k + 1, p11t, p12t, p22t, cur);
        if (nodes) memcpy(nodes + 3 * (k + 1), cur, 12);
        if (coefs) {
            float s1 = 0, c0 = 0, c2 = 0;
            if (k + 1 <= K) r32_coef(&st, r32_step(g), k + 1, p11t, p12t, p22t, &s1, &c0, &c2);
            coefs[2 * (k + 1)] = c0;
            coefs[2 * (k + 1) + 1] = c2;
        }
        const float dx = cur[0] - prev[0], dy = cur[1] - prev[1], dz = cur[2] - prev[2];
        const float len = sqrtf(fmaf(dz, dz, fmaf(dy, dy, dx * dx)));
        int32_t pv[ORC_MAX_CUTS + 1];
        float pl[ORC_MAX_CUTS + 1];
        int np = 1;
        if (g_walk_mode == 1) {
            np = r32_pieces(g, prev, cur, len, pv, pl);
        } else {
            pv[0] = r32_voxel(g, fmaf(0.5f * (prev[0] + cur[0]), inv_h, hx), fmaf(0.5f * (prev[1] + cur[1]), inv_h, hy),
                              fmaf(0.5f * (prev[2] + cur[2]), inv_h, hz));
            pl[0] = len;
        }
        if (ns + np > max_seg) return -(ns + np);
        for (int j = 0; j < np; ++j, ++ns) {
            const int32_t lin = pv[j];
            if (seg_idx) seg_idx[ns] = lin;
            if (seg_len) seg_len[ns] = pl[j];
            if (lin >= 0) {
                if (lin == last) {
                    /* merged in double by the callers that need it; here in fp32 for the debug row */
                    if (row_len) row_len[nnz - 1] += pl[j];
                } else {
                    if (row_idx) row_idx[nnz] = lin;
                    if (row_len) row_len[nnz] = pl[j];
                    ++nnz;
                }
            }
            last = lin;
        }
        memcpy(prev, cur, 12);
    }
    if (nseg_out) *nseg_out = ns;
    return nnz;
}

/* ==========================================================================================
 * DROP (R12-R18; Fig. 1): for each block, from the SAME x,
 *   r_i = (b_i - a_i.x)/||a_i||^2,  Delta_j += r_i a_ij,  c_j += 1 (j in row i)
 * then x_j += lambda Delta_j / max(1, c_j).  Rows from T32, all sums in fp64.
 * ======================================================================================== */
typedef struct {
    const float *t_in, *v_in, *t_out, *v_out, *tht_in, *thv_in, *tht_out, *thv_out, *wepl;
    const uint16_t *proj;
    const float *proj_cos, *proj_sin;
    int n_proj;
} orc_histories;

static void load_hist(const orc_histories *H, int64_t i, orc_hist *hh) {
    hh->t_in = H->t_in[i]; hh->v_in = H->v_in[i]; hh->t_out = H->t_out[i]; hh->v_out = H->v_out[i];
    hh->tht_in = H->tht_in[i]; hh->thv_in = H->thv_in[i];
    hh->tht_out = H->tht_out[i]; hh->thv_out = H->thv_out[i];
    int p = H->proj[i];
    if (p >= H->n_proj) p = H->n_proj - 1; /* DESIGN.md R24: an index past the tables means the last angle (never read out of bounds) */
    hh->cs = H->proj_cos[p];
    hh->sn = H->proj_sin[p];
}

/* Merged row of history i with fp64 lengths.  Returns nnz. */
static int row_f64(const orc_geom *g, const orc_histories *H, int64_t i, const float *p11t,
                   const float *p12t, const float *p22t, int max_seg, int32_t *sidx, float *slen,
                   int32_t *ridx, double *rlen, int *nseg_out) {
    orc_hist hh;
    int nseg = 0;
    load_hist(H, i, &hh);
    int r = orc_row_f32(g, &hh, p11t, p12t, p22t, max_seg, NULL, NULL, sidx, slen, NULL, NULL, &nseg);
    *nseg_out = nseg;
    if (r <= 0) return 0;
    int nnz = 0;
    int32_t last = -1;
    for (int k = 0; k < nseg; ++k) {
        if (sidx[k] >= 0) {
            if (sidx[k] == last) rlen[nnz - 1] += (double)slen[k];
            else { ridx[nnz] = sidx[k]; rlen[nnz] = (double)slen[k]; ++nnz; }
        }
        last = sidx[k];
    }
    return nnz;
}

/* Delta and c of ONE block [first, first+count) against image x (M doubles), no update.
 * delta (M doubles) and cnt (M int32) are overwritten.  stats (optional, 3 int64): rows with
 * nnz>0, total nnz, total raw segments.  Two phases: rows + residuals in parallel over
 * histories (read-only x), then a serial scatter in history order (deterministic). */
int orc_block_accumulate(const orc_geom *g, const orc_histories *H, int64_t first, int64_t count,
                         const double *x, double *delta, int32_t *cnt, int64_t *stats,
                         int nthreads) {
    const int nmin = orc_kmax(g); /* (most interior nodes a path can have) */
    const int max_seg = orc_row_capacity(g);
    const int64_t M = (int64_t)g->nx * g->ny * g->nz;
    float *p11t = (float *)malloc(sizeof(float) * (nmin + 1));
    float *p12t = (float *)malloc(sizeof(float) * (nmin + 1));
    float *p22t = (float *)malloc(sizeof(float) * (nmin + 1));
    int32_t *ridx = (int32_t *)malloc(sizeof(int32_t) * (size_t)count * max_seg);
    double *rlen = (double *)malloc(sizeof(double) * (size_t)count * max_seg);
    int32_t *rnnz = (int32_t *)malloc(sizeof(int32_t) * (size_t)count);
    double *res = (double *)malloc(sizeof(double) * (size_t)count);
    if (!p11t || !p12t || !p22t || !ridx || !rlen || !rnnz || !res) return -2;
    orc_sigma1_table(r32_step(g), nmin, p11t, p12t, p22t);
    int64_t nseg_total = 0;
#ifdef _OPENMP
    if (nthreads > 0) omp_set_num_threads(nthreads);
#endif
#pragma omp parallel reduction(+ : nseg_total)
    {
        int32_t *sidx = (int32_t *)malloc(sizeof(int32_t) * max_seg);
        float *slen = (float *)malloc(sizeof(float) * max_seg);
#pragma omp for schedule(dynamic, 64)
        for (int64_t r = 0; r < count; ++r) {
            int32_t *ri = ridx + (size_t)r * max_seg;
            double *rl = rlen + (size_t)r * max_seg;
            int nseg = 0;
            int nnz = row_f64(g, H, first + r, p11t, p12t, p22t, max_seg, sidx, slen, ri, rl, &nseg);
            nseg_total += nseg;
            rnnz[r] = nnz;
            res[r] = 0.0;
            if (nnz > 0) {
                double p = 0.0, n2 = 0.0;
                for (int e = 0; e < nnz; ++e) {
                    p += rl[e] * x[ri[e]];
                    n2 += rl[e] * rl[e];
                }
                res[r] = ((double)H->wepl[first + r] - p) / n2;
            }
        }
        free(sidx);
        free(slen);
    }
    memset(delta, 0, sizeof(double) * (size_t)M);
    memset(cnt, 0, sizeof(int32_t) * (size_t)M);
    int64_t rows = 0, nnz_total = 0;
    for (int64_t r = 0; r < count; ++r) {
        const int32_t *ri = ridx + (size_t)r * max_seg;
        const double *rl = rlen + (size_t)r * max_seg;
        if (rnnz[r] > 0) ++rows;
        nnz_total += rnnz[r];
        for (int e = 0; e < rnnz[r]; ++e) {
            delta[ri[e]] += res[r] * rl[e];
            cnt[ri[e]] += 1;
        }
    }
    if (stats) { stats[0] = rows; stats[1] = nnz_total; stats[2] = nseg_total; }
    free(p11t); free(p12t); free(p22t); free(ridx); free(rlen); free(rnnz); free(res);
    return 0;
}

/* n_iter sweeps of DROP over histories [0,n) in blocks of block_size, x (M doubles) in/out.
 * stats (optional, 2 int64): non-empty rows and nnz summed over the LAST sweep. */
int orc_drop_iterate(const orc_geom *g, const orc_histories *H, int64_t n, double lambda,
                     int64_t block_size, int n_iter, double *x, int64_t *stats, int nthreads) {
    const int64_t M = (int64_t)g->nx * g->ny * g->nz;
    if (n <= 0 || block_size <= 0 || n_iter < 0) return -1;
    double *delta = (double *)malloc(sizeof(double) * (size_t)M);
    int32_t *cnt = (int32_t *)malloc(sizeof(int32_t) * (size_t)M);
    if (!delta || !cnt) return -2;
    for (int it = 0; it < n_iter; ++it) {
        int64_t rows = 0, nnz = 0;
        for (int64_t first = 0; first < n; first += block_size) {
            int64_t count = n - first < block_size ? n - first : block_size;
            int64_t st[3];
            int rc = orc_block_accumulate(g, H, first, count, x, delta, cnt, st, nthreads);
            if (rc) { free(delta); free(cnt); return rc; }
            rows += st[0];
            nnz += st[1];
            for (int64_t j = 0; j < M; ++j) {
                int32_t c = cnt[j] > 1 ? cnt[j] : 1;
                x[j] += lambda * delta[j] / (double)c;
            }
        }
        if (stats) { stats[0] = rows; stats[1] = nnz; }
    }
    free(delta);
    free(cnt);
    return 0;
}

/* CARP (section 2.2 and Fig. 2; readings R27-R29), n_iter iterations, x (M doubles)
 * in/out.  "The data are ... distributed among a user-determined number of blocks (strings in CARP
 * terminology) ... we proceed to get a new estimate x_n for each data subset n using the same initial guess
 * x_0.  A new solution is then computed from the average of the different string solutions ... if a new
 * iteration is desired, the initial solution for all the subsets will be this average."
 *   strings   string p = histories [floor(p n / P), floor((p+1) n / P)) of the caller's order (R27)
 *   estimate  one sweep of the block iteration of section 2.1 over the string's histories, in blocks of
 *             block_size counted from the string's first history, starting from the common x_0 (R28)
 *   average   the arithmetic mean of the P string solutions, voxel by voxel (R29)                         */
int orc_carp_iterate(const orc_geom *g, const orc_histories *H, int64_t n, double lambda, int64_t block_size,
                     int n_iter, int n_strings, double *x, int nthreads) {
    const int64_t M = (int64_t)g->nx * g->ny * g->nz;
    if (n <= 0 || block_size <= 0 || n_iter < 0 || n_strings < 1 || n_strings > n) return -1;
    double *delta = (double *)malloc(sizeof(double) * (size_t)M);
    double *xs = (double *)malloc(sizeof(double) * (size_t)M);
    double *sum = (double *)malloc(sizeof(double) * (size_t)M);
    int32_t *cnt = (int32_t *)malloc(sizeof(int32_t) * (size_t)M);
    int rc = (!delta || !xs || !sum || !cnt) ? -2 : 0;
    for (int it = 0; it < n_iter && rc == 0; ++it) {
        for (int64_t j = 0; j < M; ++j) sum[j] = 0.0;
        for (int p = 0; p < n_strings && rc == 0; ++p) {
            const int64_t lo = (int64_t)(((__int128)p * n) / n_strings), hi = (int64_t)(((__int128)(p + 1) * n) / n_strings);
            for (int64_t j = 0; j < M; ++j) xs[j] = x[j];
            for (int64_t first = lo; first < hi && rc == 0; first += block_size) {
                const int64_t count = hi - first < block_size ? hi - first : block_size;
                int64_t st[3];
                rc = orc_block_accumulate(g, H, first, count, xs, delta, cnt, st, nthreads);
                if (rc) break;
                for (int64_t j = 0; j < M; ++j) {
                    const int32_t c = cnt[j] > 1 ? cnt[j] : 1;
                    xs[j] += lambda * delta[j] / (double)c;
                }
            }
            for (int64_t j = 0; j < M; ++j) sum[j] += xs[j];
        }
        if (rc == 0)
            for (int64_t j = 0; j < M; ++j) x[j] = sum[j] / (double)n_strings;
    }
    free(delta); free(xs); free(sum); free(cnt);
    return rc;
}

int orc_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ==========================================================================================
 * Object-frame entry point (R32): a history given as tracker HITS
 * (x, y, z) in the object frame plus its beam-frame slopes.  The hit is carried along its straight
 * ray (air, R7) to the tracker plane of the rule:
 *     u = fma(y, cos, -(x sin));  t = fma(x, cos, y sin)          (rotation about z by -phi, R8)
 *     t_pl = fma(theta_t, u_pl - u, t);  v_pl = fma(theta_v, u_pl - u, z)
 * fp32, this operation order (it feeds the rule that decides voxel indices).  *_f64: the same in
 * double, the definition the pins check.
 * ======================================================================================== */
void orc_xyz_to_beam_f32(float u_pl, int n, const float *x, const float *y, const float *z, const float *tht,
                         const float *thv, const uint16_t *proj, const float *pcos, const float *psin, int n_proj,
                         float *t_out, float *v_out) {
    for (int i = 0; i < n; ++i) {
        int p = proj[i];
        if (p >= n_proj) p = n_proj - 1; /* R24 */
        const float cs = pcos[p], sn = psin[p];
        const float u = fmaf(y[i], cs, -(x[i] * sn));
        const float t = fmaf(x[i], cs, y[i] * sn);
        const float du = u_pl - u;
        t_out[i] = fmaf(tht[i], du, t);
        v_out[i] = fmaf(thv[i], du, z[i]);
    }
}
void orc_xyz_to_beam_f64(double u_pl, double x, double y, double z, double tht, double thv, double cs, double sn,
                         double out[2]) {
    const double u = -x * sn + y * cs, t = x * cs + y * sn;
    out[0] = t + tht * (u_pl - u);
    out[1] = z + thv * (u_pl - u);
}

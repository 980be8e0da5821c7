/*
 * mmc_oracle.c -- plain fp64 CPU oracle for the micromagnetic Monte Carlo (MMC) hot path of
 * arXiv:2106.05593 (S. Lepadatu).  TEST INFRASTRUCTURE ONLY: nothing on the product path may
 * import, link or call this file (only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs do).  It shares no code with the CUDA library.
 *
 * Every function cites the passage of /root/reference/PAPER.md (by line, section, equation) or
 * the SURVEY.md section 8(c) reading (O1..O8, G1..G15) it follows.  The arithmetic is written in
 * the paper's order and notation, one cell at a time, no blocking, no fusion.
 *
 * Cell index c = i + nx*(j + ny*k), x fastest.  m = M/Ms0.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#include <quadmath.h>

#define ORC_KB   1.380649e-23            /* J/K   */
#define ORC_MU0  (4.0e-7 * M_PI)         /* T m/A */

/* ------------------------------------------------------------------------------------------ */
/* O2. Philox4x32-10 (paper is silent on the RNG; north_star (b)).             */
/* Round: hi,lo = 0xD2511F53*c0 ; hi',lo' = 0xCD9E8D57*c2 ;                                    */
/*        c <- (hi'^c1^k0, lo', hi^c3^k1, lo) ; k <- (k0+0x9E3779B9, k1+0xBB67AE85); 10 rounds. */
/* ------------------------------------------------------------------------------------------ */
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int r = 0; r < 10; ++r) {
        uint64_t p0 = (uint64_t)0xD2511F53u * (uint64_t)c0;
        uint64_t p1 = (uint64_t)0xCD9E8D57u * (uint64_t)c2;
        uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
        uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
        uint32_t n0 = hi1 ^ c1 ^ k0;
        uint32_t n1 = lo1;
        uint32_t n2 = hi0 ^ c3 ^ k1;
        uint32_t n3 = lo0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* u = ((x>>9)+0.5)*2^-23 : strictly inside (0,1), exactly representable in fp32 (O2). */
double orc_u01(uint32_t x) { return ((double)(x >> 9) + 0.5) * (1.0 / 8388608.0); }

/* The four uniforms of cell c in sweep s: key=(seed lo, seed hi), ctr=(c lo, c hi, s lo, s hi). */
void orc_cell_uniforms(uint64_t seed, uint64_t sweep, uint64_t cell, double u[4])
{
    uint32_t key[2] = { (uint32_t)seed, (uint32_t)(seed >> 32) };
    uint32_t ctr[4] = { (uint32_t)cell, (uint32_t)(cell >> 32), (uint32_t)sweep, (uint32_t)(sweep >> 32) };
    uint32_t x[4];
    orc_philox4x32_10(ctr, key, x);
    for (int a = 0; a < 4; ++a) u[a] = orc_u01(x[a]);
}

/* ------------------------------------------------------------------------------------------ */
/* O1. Thermal parameterisation: Eq. (8), (9), (7), (13) -- PAPER.md:62-72, 104-106.           */
/* ------------------------------------------------------------------------------------------ */
/* Langevin function B(x) = coth x - 1/x.  coth x - 1/x cancels like 1/x^2 for small x,
   so |x| < 0.1 uses the Taylor series x/3 - x^3/45 + 2x^5/945 - x^7/4725 + 2x^9/93555 (next term 2e-17). */
double orc_langevin(double x)
{
    if (fabs(x) < 0.1) {
        double x2 = x * x;
        return x * (1.0 / 3.0 + x2 * (-1.0 / 45.0 + x2 * (2.0 / 945.0 + x2 * (-1.0 / 4725.0 + x2 * (2.0 / 93555.0)))));
    }
    return 1.0 / tanh(x) - 1.0 / x;
}
/* B'(x) = 1/x^2 - 1/sinh^2 x, B'(0) = 1/3; derivative of the series above for |x| < 0.1. */
double orc_langevin_prime(double x)
{
    if (fabs(x) < 0.1) {
        double x2 = x * x;
        return 1.0 / 3.0 + x2 * (-3.0 / 45.0 + x2 * (10.0 / 945.0 + x2 * (-7.0 / 4725.0 + x2 * (18.0 / 93555.0))));
    }
    if (fabs(x) > 350.0) return 1.0 / (x * x);
    double sh = sinh(x);
    return 1.0 / (x * x) - 1.0 / (sh * sh);
}
/* Eq. (9) with H_ext = 0 (reading G3): me = B(me*3Tc/T); me = 0 for T >= Tc.  Bisection. */
double orc_me(double T, double Tc)
{
    if (!(T < Tc)) return 0.0;
    double a = 3.0 * Tc / T;
    double lo = 0.0, hi = 1.0;               /* g(me) = B(a me) - me: >0 just above 0, <0 at 1 */
    for (int it = 0; it < 200; ++it) {
        double mid = 0.5 * (lo + hi);
        if (orc_langevin(a * mid) - mid > 0.0) lo = mid; else hi = mid;
    }
    return 0.5 * (lo + hi);
}
/* Eq. (8): chi~ = (mu/kB T) B'(x)/(1 - B'(x) 3Tc/T), x = me 3Tc/T.  Units 1/tesla. */
double orc_chi_par(double T, double Tc, double mu, double me)
{
    double a = 3.0 * Tc / T, x = me * a;
    double bp = orc_langevin_prime(x);
    return (mu / (ORC_KB * T)) * bp / (1.0 - bp * a);
}
/*
 * Longitudinal free energy in units of kB T as a quartic  F_l/kBT = c4 m^4 + c2 m^2 + c0
 * (exponent of Eq. (7)):
 *   T<Tc: c = V Ms0/(8 chi~ me^2 kB T); c4 = c, c2 = -2 c me^2, c0 = c me^4
 *   T>Tc: c2 = V Ms0/(2 chi~ kB T);    c4 = c2 * 3Tc/(10 (T-Tc)), c0 = 0
 *   |T-Tc|/Tc < 1e-7 (reading G10): common limit c2 = 0, c4 = (9/20) V Ms0/mu, c0 = 0.
 * sigma13 = Eq. (13) capped at 0.03, constant 0.03 for T >= Tc.
 * out = {me, chi, c2, c4, c0, sigma13}.  Returns 0, or -1 if T <= 0.
 */
int orc_thermal(double T, double Tc, double mu, double V, double Ms0, double out[6])
{
    if (!(T > 0.0)) return -1;
    double me, chi, c2, c4, c0, sg;
    if (fabs(T - Tc) < 1e-7 * Tc) {
        me = 0.0; chi = INFINITY; c2 = 0.0; c4 = (9.0 / 20.0) * V * Ms0 / mu; c0 = 0.0; sg = 0.03;
    } else if (T < Tc) {
        me = orc_me(T, Tc);
        chi = orc_chi_par(T, Tc, mu, me);
        double c = V * Ms0 / (8.0 * chi * me * me * ORC_KB * T);
        c4 = c; c2 = -2.0 * c * me * me; c0 = c * me * me * me * me;
        sg = 2.0 * me * sqrt(chi * ORC_KB * T / (V * Ms0));
        if (sg > 0.03) sg = 0.03;
    } else {
        me = 0.0;
        chi = orc_chi_par(T, Tc, mu, 0.0);
        c2 = V * Ms0 / (2.0 * chi * ORC_KB * T);
        c4 = c2 * 3.0 * Tc / (10.0 * (T - Tc));
        c0 = 0.0; sg = 0.03;
    }
    out[0] = me; out[1] = chi; out[2] = c2; out[3] = c4; out[4] = c0; out[5] = sg;
    return 0;
}

/* ------------------------------------------------------------------------------------------ */
/* Problem description: per-cell coefficient arrays, filled by the Python side from orc_thermal */
/* ------------------------------------------------------------------------------------------ */
typedef struct {
    int32_t nx, ny, nz;
    uint32_t pbc;                 /* bit0 = x, bit1 = y, bit2 = z */
    double dx, dy, dz;            /* cell edges, m */
    const uint8_t *active;        /* N: 1 where Ms0 > 0 */
    const int32_t *region;        /* N: region id */
    int32_t inter_region_exchange;/* 0: bonds between different regions carry no exchange/DMI */
    const double *Ms0;            /* N, A/m */
    const double *beta;           /* N, 1/(kB T_c) */
    const double *c2, *c4, *c0;   /* N, longitudinal quartic in units of kB T */
    const double *Kq;             /* N, K1,0 * me  (J/m^3), 0 for T >= Tc (reading G5) */
    const double *K1T;            /* N, K1(T) = K1,0 * me^3 (for the E_an read-out constant) */
    const double *ax, *ay, *az;   /* N, unit easy axis */
    const double *sigma;          /* N, half-width of the length factor */
    double A0, D0;                /* J/m, J/m^2 -- uniform over non-empty cells */
    double Bext[3];               /* tesla */
    const double *bdx, *bdy, *bdz;/* N each, frozen B_d = mu0 H_d (tesla); NULL = no demag */
    double one_minus_cos_cone;    /* 1 - cos(theta_c) */
    uint64_t seed;
    /* cubic anisotropy, Eq. (12): NULL = none */
    const double *K1cT, *K2cT;    /* N, K1c me^10 and K2c me^21 (me^(l(l+1)/2), l = 4, 6), 0 for T >= Tc */
    const double *cub;            /* 9N: the three orthonormal cubic axes of the cell, cub[9c + 3a + q] */
    /* 4th-order uniaxial term of Eq. (11), reading G5 (m_i there = M/Ms(T) = m/me): NULL = none */
    const double *K2T;            /* N, K2 me^10 (l = 4 in me^(l(l+1)/2)), 0 for T >= Tc */
    const double *me2;            /* N, me^2 */
} orc_problem;

/* Eq. (12): alpha^2 beta^2 + alpha^2 gamma^2 + beta^2 gamma^2 and alpha^2 beta^2 gamma^2 of the DIRECTION of v          */
/* ("direction cosines of the magnetization vector") with respect to the cell's cubic axes.                */
static void orc_cubic_invariants(const double *ax9, const double v[3], double *c1, double *c2)
{
    double L = sqrt(v[0] * v[0] + v[1] * v[1] + v[2] * v[2]);
    double a = (v[0] * ax9[0] + v[1] * ax9[1] + v[2] * ax9[2]) / L;
    double b = (v[0] * ax9[3] + v[1] * ax9[4] + v[2] * ax9[5]) / L;
    double g = (v[0] * ax9[6] + v[1] * ax9[7] + v[2] * ax9[8]) / L;
    *c1 = a * a * b * b + a * a * g * g + b * b * g * g;
    *c2 = a * a * b * b * g * g;
}

static inline int64_t orc_idx(const orc_problem *p, int i, int j, int k)
{
    return (int64_t)i + (int64_t)p->nx * ((int64_t)j + (int64_t)p->ny * (int64_t)k);
}

/*
 * Neighbour of (i,j,k) in direction d (0:+x 1:-x 2:+y 3:-y 4:+z 5:-z); -1 if it does not exist.
 * Periodic wrap where the pbc bit is set (O6: periodic lengths are even, checked by the caller).
 * "bonded" (O4, G9): exists, non-empty, and in the same region unless inter-region exchange on.
 */
static int64_t orc_neighbour(const orc_problem *p, int i, int j, int k, int d)
{
    int n[3] = { p->nx, p->ny, p->nz };
    int q[3] = { i, j, k };
    int a = d >> 1, step = (d & 1) ? -1 : +1;
    int v = q[a] + step;
    if (v < 0 || v >= n[a]) {
        if (!((p->pbc >> a) & 1u) || n[a] < 2) return -1;
        v = (v + n[a]) % n[a];
    }
    q[a] = v;
    return orc_idx(p, q[0], q[1], q[2]);
}
static int orc_bonded(const orc_problem *p, int64_t c, int64_t nb)
{
    if (nb < 0) return 0;
    if (!p->active[nb]) return 0;
    if (!p->inter_region_exchange && p->region[nb] != p->region[c]) return 0;
    return 1;
}

/* ------------------------------------------------------------------------------------------ */
/* O3. Trial move (PAPER.md:92 steps 1-2; readings G6).                          */
/*   u = (u_cos, u_phi, u_len).  Outputs dm (3) and f = |m'|/|m| = 1 + s.                      */
/* ------------------------------------------------------------------------------------------ */
void orc_trial(const double m[3], const double u[3], double one_minus_cos_cone, double sigma,
               double dm[3], double *f_out)
{
    double L = sqrt(m[0] * m[0] + m[1] * m[1] + m[2] * m[2]);
    double n[3] = { m[0] / L, m[1] / L, m[2] / L };
    /* a = coordinate axis with the smallest |m_a| (raw stored components, ties -> lowest index) */
    int a = 0;
    if (fabs(m[1]) < fabs(m[a])) a = 1;
    if (fabs(m[2]) < fabs(m[a])) a = 2;
    double t1[3], t2[3];
    if (a == 0)      { t1[0] = 0.0;   t1[1] = -n[2]; t1[2] = n[1]; }   /* e_x x n */
    else if (a == 1) { t1[0] = n[2];  t1[1] = 0.0;   t1[2] = -n[0]; }  /* e_y x n */
    else             { t1[0] = -n[1]; t1[1] = n[0];  t1[2] = 0.0; }    /* e_z x n */
    double tl = sqrt(t1[0] * t1[0] + t1[1] * t1[1] + t1[2] * t1[2]);
    t1[0] /= tl; t1[1] /= tl; t1[2] /= tl;
    t2[0] = n[1] * t1[2] - n[2] * t1[1];                               /* t2 = n x t1 */
    t2[1] = n[2] * t1[0] - n[0] * t1[2];
    t2[2] = n[0] * t1[1] - n[1] * t1[0];
    double w = u[0] * one_minus_cos_cone;          /* omega = 1 - cos(theta): uniform on the cap */
    double st = sqrt(w * (2.0 - w));
    double phi = 2.0 * M_PI * u[1];
    double cp = cos(phi), sp = sin(phi);
    double dn[3];
    for (int q = 0; q < 3; ++q) dn[q] = st * (cp * t1[q] + sp * t2[q]) - w * n[q];
    double s = sigma * (2.0 * u[2] - 1.0);         /* f = 1 + s in [1-sigma, 1+sigma] */
    for (int q = 0; q < 3; ++q) dm[q] = L * ((1.0 + s) * dn[q] + s * n[q]);
    *f_out = 1.0 + s;
}

/* ------------------------------------------------------------------------------------------ */
/* O4. Local free-energy change in units of kB T_c for trial dm on cell (i,j,k).               */
/* terms = { ex, an, zee, dmi, demag, long }.                                                   */
/*  ex   : Eq. (10) with the factor 2, reading G2 (exact change of the pair    */
/*         energy): -beta sum_d J_d dm.sum_{nb bonded}(m_nb - m) + beta (sum_d J_d n_d/2)|dm|^2 */
/*         J_d = 2 A0 V/h_d^2                                                                   */
/*  an   : Eq. (11) K1 term, reading G5: -beta V Kq (dm.e)((2m+dm).e)                           */
/*  zee  : "applied field": -beta V Ms0 dm.B_ext                                  */
/*  demag: Eq. (14): -beta V Ms0 dm.B_d with B_d frozen for the pass         */
/*  dmi  : Eq. (15), literal sign (G7): -beta 2 D0 V dm.G,                       */
/*         G = 1/2 ( -(mzE-mzW)/dx, -(mzN-mzS)/dy, (mxE-mxW)/dx + (myN-myS)/dy ),               */
/*         an unbonded neighbour contributes 0 (G8)                                             */
/*  long : exponent of Eq. (7) (PAPER.md:62, 92 step 3): dl2 (c4 (l2' + l2) + c2)               */
/* ------------------------------------------------------------------------------------------ */
void orc_cell_dF(const orc_problem *p, const double *mx, const double *my, const double *mz,
                 int i, int j, int k, const double dm[3], double terms[6])
{
    int64_t c = orc_idx(p, i, j, k);
    double V = p->dx * p->dy * p->dz;
    double h[3] = { p->dx, p->dy, p->dz };
    double beta = p->beta[c];
    double m[3] = { mx[c], my[c], mz[c] };
    double mn[6][3]; int bond[6];
    for (int d = 0; d < 6; ++d) {
        int64_t nb = orc_neighbour(p, i, j, k, d);
        bond[d] = orc_bonded(p, c, nb);
        if (bond[d]) { mn[d][0] = mx[nb]; mn[d][1] = my[nb]; mn[d][2] = mz[nb]; }
        else         { mn[d][0] = mn[d][1] = mn[d][2] = 0.0; }
    }
    /* exchange */
    double ex_lin = 0.0, ex_self = 0.0;
    for (int a = 0; a < 3; ++a) {
        double Jd = 2.0 * p->A0 * V / (h[a] * h[a]);
        int nd = 0; double S[3] = { 0, 0, 0 };
        for (int s = 0; s < 2; ++s) {
            int d = 2 * a + s;
            if (!bond[d]) continue;
            nd++;
            for (int q = 0; q < 3; ++q) S[q] += mn[d][q] - m[q];
        }
        ex_lin += Jd * (dm[0] * S[0] + dm[1] * S[1] + dm[2] * S[2]);
        ex_self += Jd * nd / 2.0;
    }
    double dm2 = dm[0] * dm[0] + dm[1] * dm[1] + dm[2] * dm[2];
    terms[0] = -beta * ex_lin + beta * ex_self * dm2;
    /* uniaxial anisotropy */
    double e[3] = { p->ax[c], p->ay[c], p->az[c] };
    double dme = dm[0] * e[0] + dm[1] * e[1] + dm[2] * e[2];
    double sme = (2 * m[0] + dm[0]) * e[0] + (2 * m[1] + dm[1]) * e[1] + (2 * m[2] + dm[2]) * e[2];
    terms[1] = -beta * V * p->Kq[c] * dme * sme;
    /* Eq. (11), second term, times V (the paper's V is missing there, G5): K2(T) [1 - (m.e)^2/me^2]^2, trial minus current */
    if (p->K2T && p->K2T[c] != 0.0) {
        double q0 = m[0] * e[0] + m[1] * e[1] + m[2] * e[2];
        double q1 = q0 + dme;
        double g0 = 1.0 - q0 * q0 / p->me2[c], g1 = 1.0 - q1 * q1 / p->me2[c];
        terms[1] += beta * V * p->K2T[c] * (g1 * g1 - g0 * g0);
    }
    /* cubic anisotropy, Eq. (12), both terms times V: the plain difference of the energy of the trial and the current direction */
    if (p->cub) {
        double mp[3] = { m[0] + dm[0], m[1] + dm[1], m[2] + dm[2] };
        double a1, a2, b1, b2;
        orc_cubic_invariants(p->cub + 9 * c, m, &a1, &a2);
        orc_cubic_invariants(p->cub + 9 * c, mp, &b1, &b2);
        terms[1] += beta * V * (p->K1cT[c] * (b1 - a1) + p->K2cT[c] * (b2 - a2));
    }
    /* Zeeman */
    double bvm = beta * V * p->Ms0[c];
    terms[2] = -bvm * (dm[0] * p->Bext[0] + dm[1] * p->Bext[1] + dm[2] * p->Bext[2]);
    /* interfacial DMI; E=+x(0) W=-x(1) N=+y(2) S=-y(3) */
    double G[3];
    G[0] = 0.5 * (-(mn[0][2] - mn[1][2]) / p->dx);
    G[1] = 0.5 * (-(mn[2][2] - mn[3][2]) / p->dy);
    G[2] = 0.5 * ((mn[0][0] - mn[1][0]) / p->dx + (mn[2][1] - mn[3][1]) / p->dy);
    terms[3] = -beta * 2.0 * p->D0 * V * (dm[0] * G[0] + dm[1] * G[1] + dm[2] * G[2]);
    /* demag, frozen field */
    if (p->bdx) terms[4] = -bvm * (dm[0] * p->bdx[c] + dm[1] * p->bdy[c] + dm[2] * p->bdz[c]);
    else        terms[4] = 0.0;
    /* longitudinal */
    double l2 = m[0] * m[0] + m[1] * m[1] + m[2] * m[2];
    double dl2 = dm[0] * (2 * m[0] + dm[0]) + dm[1] * (2 * m[1] + dm[1]) + dm[2] * (2 * m[2] + dm[2]);
    double l2p = l2 + dl2;
    terms[5] = dl2 * (p->c4[c] * (l2p + l2) + p->c2[c]);
}

/* ------------------------------------------------------------------------------------------ */
/* O5 + O6. One colour pass (PAPER.md:92 steps 1-4, checkerboard; Eq. (5)).        */
/*  Visits every active cell with (i+j+k)%2 == colour exactly once, in lexicographic order, or  */
/*  in the order given by `order` (a list of n_order cell indices of that colour; used by the   */
/*  order-independence pin).  Accept iff ln u_acc < 4 ln f - dF/kBT (strict, G14; G1 literal).  */
/*  store_fp32 != 0 rounds an accepted m' to fp32 (the state's storage format on the GPU).      */
/*  Optional per-cell dumps (may be NULL): dm_out[3N], terms_out[6N], margin_out[N], acc_out[N].*/
/*  Returns accepted count; *trials_out = number of cells that received a trial.                */
/* ------------------------------------------------------------------------------------------ */
static int orc_visit(const orc_problem *p, double *mx, double *my, double *mz, int i, int j, int k,
                     uint64_t sweep, int store_fp32,
                     double *dm_out, double *terms_out, double *margin_out, uint8_t *acc_out)
{
    int64_t c = orc_idx(p, i, j, k);
    double u[4];
    orc_cell_uniforms(p->seed, sweep, (uint64_t)c, u);
    double m[3] = { mx[c], my[c], mz[c] };
    double dm[3], f, terms[6];
    orc_trial(m, u, p->one_minus_cos_cone, p->sigma[c], dm, &f);
    orc_cell_dF(p, mx, my, mz, i, j, k, dm, terms);
    double dF = terms[0] + terms[1] + terms[2] + terms[3] + terms[4] + terms[5];
    double margin = log(u[3]) - 4.0 * log(f) + dF;       /* accept <=> margin < 0 */
    int acc = margin < 0.0;
    if (dm_out)     { dm_out[3 * c] = dm[0]; dm_out[3 * c + 1] = dm[1]; dm_out[3 * c + 2] = dm[2]; }
    if (terms_out)  for (int q = 0; q < 6; ++q) terms_out[6 * c + q] = terms[q];
    if (margin_out) margin_out[c] = margin;
    if (acc_out)    acc_out[c] = (uint8_t)acc;
    if (acc) {
        double a = m[0] + dm[0], b = m[1] + dm[1], d = m[2] + dm[2];
        if (store_fp32) { a = (double)(float)a; b = (double)(float)b; d = (double)(float)d; }
        mx[c] = a; my[c] = b; mz[c] = d;
    }
    return acc;
}

int64_t orc_colour_pass(const orc_problem *p, double *mx, double *my, double *mz, int colour,
                        uint64_t sweep, const int64_t *order, int64_t n_order, int store_fp32,
                        double *dm_out, double *terms_out, double *margin_out, uint8_t *acc_out,
                        int64_t *trials_out)
{
    int64_t accepted = 0, trials = 0;
    if (order) {
        for (int64_t q = 0; q < n_order; ++q) {
            int64_t c = order[q];
            int i = (int)(c % p->nx), j = (int)((c / p->nx) % p->ny), k = (int)(c / ((int64_t)p->nx * p->ny));
            if (((i + j + k) & 1) != colour || !p->active[c]) continue;
            trials++;
            accepted += orc_visit(p, mx, my, mz, i, j, k, sweep, store_fp32, dm_out, terms_out, margin_out, acc_out);
        }
    } else {
        /* cells of one colour never read each other (6-stencil and DMI E/W/N/S are all of the
           other colour), so the rows may be visited by several threads: same result (O6). */
        #pragma omp parallel for collapse(2) reduction(+:accepted, trials) schedule(static)
        for (int k = 0; k < p->nz; ++k)
            for (int j = 0; j < p->ny; ++j)
                for (int i = (j + k + colour) & 1; i < p->nx; i += 2) {
                    int64_t c = orc_idx(p, i, j, k);
                    if (!p->active[c]) continue;
                    trials++;
                    accepted += orc_visit(p, mx, my, mz, i, j, k, sweep, store_fp32, dm_out, terms_out, margin_out, acc_out);
                }
    }
    if (trials_out) *trials_out = trials;
    return accepted;
}

/* ------------------------------------------------------------------------------------------ */
/* O8. Read-outs.  Energies in joule, pair terms counted once.                                 */
/*  out = { E_ex, E_an, E_zee, E_dmi, E_demag, E_long },                                        */
/*  E_ex = sum_bonds (A0 V/h_d^2)|m_i-m_j|^2 ; E_dmi = -D0 V sum_i m_i.G_i ;                     */
/*  E_an = sum V [K1(T) - Kq (m.e)^2] ; E_zee = -V sum Ms0 m.B_ext ;                             */
/*  E_demag = -(V/2) sum Ms0 m.B_d ; E_long = sum kB T (c4 m^4 + c2 m^2 + c0).                   */
/*  mean = { <mx>, <my>, <mz>, <|m|> } over active cells.                                        */
/* ------------------------------------------------------------------------------------------ */
void orc_observables(const orc_problem *p, const double *mx, const double *my, const double *mz,
                     double out[6], double mean[4], int64_t *n_active)
{
    double V = p->dx * p->dy * p->dz;
    double h[3] = { p->dx, p->dy, p->dz };
    double Eex = 0, Ean = 0, Ezee = 0, Edmi = 0, Edem = 0, Elong = 0;
    double sx = 0, sy = 0, sz = 0, sl = 0; int64_t na = 0;
    for (int k = 0; k < p->nz; ++k)
    for (int j = 0; j < p->ny; ++j)
    for (int i = 0; i < p->nx; ++i) {
        int64_t c = orc_idx(p, i, j, k);
        if (!p->active[c]) continue;
        double m[3] = { mx[c], my[c], mz[c] };
        na++; sx += m[0]; sy += m[1]; sz += m[2];
        double l2 = m[0] * m[0] + m[1] * m[1] + m[2] * m[2];
        sl += sqrt(l2);
        double mn[6][3]; int bond[6];
        for (int d = 0; d < 6; ++d) {
            int64_t nb = orc_neighbour(p, i, j, k, d);
            bond[d] = orc_bonded(p, c, nb);
            if (bond[d]) { mn[d][0] = mx[nb]; mn[d][1] = my[nb]; mn[d][2] = mz[nb]; }
            else         { mn[d][0] = mn[d][1] = mn[d][2] = 0.0; }
        }
        /* each bond is seen from both ends: half weight here counts it once */
        for (int d = 0; d < 6; ++d) if (bond[d]) {
            double a0 = m[0] - mn[d][0], a1 = m[1] - mn[d][1], a2 = m[2] - mn[d][2];
            Eex += 0.5 * (p->A0 * V / (h[d >> 1] * h[d >> 1])) * (a0 * a0 + a1 * a1 + a2 * a2);
        }
        double G[3];
        G[0] = 0.5 * (-(mn[0][2] - mn[1][2]) / p->dx);
        G[1] = 0.5 * (-(mn[2][2] - mn[3][2]) / p->dy);
        G[2] = 0.5 * ((mn[0][0] - mn[1][0]) / p->dx + (mn[2][1] - mn[3][1]) / p->dy);
        Edmi += -p->D0 * V * (m[0] * G[0] + m[1] * G[1] + m[2] * G[2]);
        double me_ = m[0] * p->ax[c] + m[1] * p->ay[c] + m[2] * p->az[c];
        Ean += V * (p->K1T[c] - p->Kq[c] * me_ * me_);
        if (p->K2T && p->K2T[c] != 0.0) { double g = 1.0 - me_ * me_ / p->me2[c]; Ean += V * p->K2T[c] * g * g; }
        if (p->cub) {
            double c1, c2;
            orc_cubic_invariants(p->cub + 9 * c, m, &c1, &c2);
            Ean += V * (p->K1cT[c] * c1 + p->K2cT[c] * c2);
        }
        Ezee += -V * p->Ms0[c] * (m[0] * p->Bext[0] + m[1] * p->Bext[1] + m[2] * p->Bext[2]);
        if (p->bdx) Edem += -0.5 * V * p->Ms0[c] * (m[0] * p->bdx[c] + m[1] * p->bdy[c] + m[2] * p->bdz[c]);
        Elong += (1.0 / p->beta[c]) * (p->c4[c] * l2 * l2 + p->c2[c] * l2 + p->c0[c]);
    }
    out[0] = Eex; out[1] = Ean; out[2] = Ezee; out[3] = Edmi; out[4] = Edem; out[5] = Elong;
    if (na > 0) { mean[0] = sx / na; mean[1] = sy / na; mean[2] = sz / na; mean[3] = sl / na; }
    else mean[0] = mean[1] = mean[2] = mean[3] = 0.0;
    if (n_active) *n_active = na;
}

/* ------------------------------------------------------------------------------------------ */
/* O7. Demagnetising tensor (paper cites [17,31] only; north_star names Newell).  */
/*  N_xx(X,Y,Z) = 1/(4 pi dx dy dz) sum_{i,j,k in -1,0,1} w_i w_j w_k f(X+i dx, Y+j dy, Z+k dz)  */
/*  with w_0 = 2, w_+-1 = -1; N_xy likewise with g; other components by permutation.             */
/*  Evaluated in binary128 (libquadmath) because the 27-point sum cancels ~(r/h)^6.              */
/* ------------------------------------------------------------------------------------------ */
typedef __float128 q128;

static q128 nw_f(q128 x, q128 y, q128 z)
{
    q128 x2 = x * x, y2 = y * y, z2 = z * z;
    q128 R = sqrtq(x2 + y2 + z2);
    q128 r = 0;
    if (y != 0 && (x2 + z2) > 0) r += (y / 2) * (z2 - x2) * asinhq(y / sqrtq(x2 + z2));
    if (z != 0 && (x2 + y2) > 0) r += (z / 2) * (y2 - x2) * asinhq(z / sqrtq(x2 + y2));
    if (x != 0 && y != 0 && z != 0) r -= x * y * z * atanq(y * z / (x * R));
    r += (2 * x2 - y2 - z2) * R / 6;
    return r;
}
static q128 nw_g(q128 x, q128 y, q128 z)
{
    q128 x2 = x * x, y2 = y * y, z2 = z * z;
    q128 R = sqrtq(x2 + y2 + z2);
    q128 r = 0;
    if (x != 0 && y != 0 && z != 0) r += x * y * z * asinhq(z / sqrtq(x2 + y2));
    if (y != 0 && x != 0) r += (y / 6) * (3 * z2 - y2) * asinhq(x / sqrtq(y2 + z2));
    if (x != 0 && y != 0) r += (x / 6) * (3 * z2 - x2) * asinhq(y / sqrtq(x2 + z2));
    if (z != 0 && x != 0 && y != 0) {
        r -= (z * z2 / 6) * atanq(x * y / (z * R));
        r -= (z * y2 / 2) * atanq(x * z / (y * R));
        r -= (z * x2 / 2) * atanq(y * z / (x * R));
    }
    r -= x * y * R / 3;
    return r;
}
static q128 nw_stencil(q128 (*fn)(q128, q128, q128), q128 X, q128 Y, q128 Z, q128 dx, q128 dy, q128 dz)
{
    q128 s = 0;
    for (int i = -1; i <= 1; ++i)
    for (int j = -1; j <= 1; ++j)
    for (int k = -1; k <= 1; ++k) {
        q128 w = (q128)((i == 0 ? 2 : -1) * (j == 0 ? 2 : -1) * (k == 0 ? 2 : -1));
        s += w * fn(X + i * dx, Y + j * dy, Z + k * dz);
    }
    return s / (4 * M_PIq * dx * dy * dz);
}
/* Newell tensor at offset (X,Y,Z) metres for cells dx*dy*dz.  out = {xx, yy, zz, xy, xz, yz}. */
void orc_newell(double X, double Y, double Z, double dx, double dy, double dz, double out[6])
{
    out[0] = (double)nw_stencil(nw_f, X, Y, Z, dx, dy, dz);
    out[1] = (double)nw_stencil(nw_f, Y, X, Z, dy, dx, dz);   /* N_yy <-> f(y,x,z) */
    out[2] = (double)nw_stencil(nw_f, Z, Y, X, dz, dy, dx);   /* N_zz <-> f(z,y,x) */
    out[3] = (double)nw_stencil(nw_g, X, Y, Z, dx, dy, dz);   /* N_xy <-> g(x,y,z) */
    out[4] = (double)nw_stencil(nw_g, X, Z, Y, dx, dz, dy);   /* N_xz <-> g(x,z,y) */
    out[5] = (double)nw_stencil(nw_g, Y, Z, X, dy, dz, dx);   /* N_yz <-> g(y,z,x) */
}
/* Point-dipole tensor of a cube of volume v at offset r: (v/4pi)(delta_ab/r^3 - 3 r_a r_b/r^5). */
static void orc_dipole(double X, double Y, double Z, double v, double out[6])
{
    double r2 = X * X + Y * Y + Z * Z, r = sqrt(r2), r3 = r2 * r, r5 = r3 * r2;
    double c = v / (4.0 * M_PI);
    out[0] = c * (1.0 / r3 - 3.0 * X * X / r5);
    out[1] = c * (1.0 / r3 - 3.0 * Y * Y / r5);
    out[2] = c * (1.0 / r3 - 3.0 * Z * Z / r5);
    out[3] = c * (-3.0 * X * Y / r5);
    out[4] = c * (-3.0 * X * Z / r5);
    out[5] = c * (-3.0 * Y * Z / r5);
}
/*
 * Far-field form: split source and target cell into px*py*pz cubes of side hc
 * (dx = px hc, ...; the configs have 1x1x1 and 1x1x2) and average the cube-cube dipole terms:
 *   N = (1/P) sum_{a in target cubes} sum_{b in source cubes} N_cube(R + r_a - r_b),  P = px py pz.
 */
static void orc_far(double X, double Y, double Z, double hc, int px, int py, int pz, double out[6])
{
    double acc[6] = { 0, 0, 0, 0, 0, 0 }, t[6];
    double v = hc * hc * hc; int P = px * py * pz;
    for (int ax = 0; ax < px; ++ax) for (int bx = 0; bx < px; ++bx)
    for (int ay = 0; ay < py; ++ay) for (int by = 0; by < py; ++by)
    for (int az = 0; az < pz; ++az) for (int bz = 0; bz < pz; ++bz) {
        orc_dipole(X + (ax - bx) * hc, Y + (ay - by) * hc, Z + (az - bz) * hc, v, t);
        for (int q = 0; q < 6; ++q) acc[q] += t[q];
    }
    for (int q = 0; q < 6; ++q) out[q] = acc[q] / P;
}
/*
 * Tensor table for offsets ox in [0,nx), oy in [0,ny), oz in [0,nz) (other octants follow from
 * the parity of each component).  out[q][(oz*ny + oy)*nx + ox], q = xx,yy,zz,xy,xz,yz.
 * Newell (binary128) when max(|ox|,|oy|,|oz|) <= r_near cells or the cell cannot be split into
 * cubes; sub-cube dipole average beyond.
 */
void orc_demag_tensor(int nx, int ny, int nz, double dx, double dy, double dz, int r_near, double *out)
{
    double hc = fmin(dx, fmin(dy, dz));
    int px = (int)lround(dx / hc), py = (int)lround(dy / hc), pz = (int)lround(dz / hc);
    int splittable = fabs(px * hc - dx) < 1e-9 * hc && fabs(py * hc - dy) < 1e-9 * hc && fabs(pz * hc - dz) < 1e-9 * hc
                     && px * py * pz <= 8;
    int64_t P = (int64_t)nx * ny * nz;
    #pragma omp parallel for collapse(2) schedule(dynamic, 8)
    for (int oz = 0; oz < nz; ++oz)
    for (int oy = 0; oy < ny; ++oy)
    for (int ox = 0; ox < nx; ++ox) {
        double t[6];
        int far = splittable && (ox > r_near || oy > r_near || oz > r_near);
        if (far) orc_far(ox * dx, oy * dy, oz * dz, hc, px, py, pz, t);
        else     orc_newell(ox * dx, oy * dy, oz * dz, dx, dy, dz, t);
        int64_t o = ((int64_t)oz * ny + oy) * nx + ox;
        for (int q = 0; q < 6; ++q) out[q * P + o] = t[q];
    }
}
/*
 * Eq. (14): H_d,i = -sum_j N(r_i - r_j) M_j by the direct O(N^2) sum, returned as
 * B_d = mu0 H_d in tesla.  Mx,My,Mz = Ms0_j m_j in A/m (0 in empty cells).  `tab` is the octant
 * table of orc_demag_tensor; N_ab(-x) = N_ab(x) for a==b, and picks up sign(ox)sign(oy) etc. for
 * the off-diagonal components.
 */
void orc_demag_direct(int nx, int ny, int nz, const double *tab,
                      const double *Mx, const double *My, const double *Mz,
                      double *bx, double *by, double *bz)
{
    int64_t P = (int64_t)nx * ny * nz;
    #pragma omp parallel for schedule(static)
    for (int64_t ci = 0; ci < P; ++ci) {
        int i = (int)(ci % nx), j = (int)((ci / nx) % ny), k = (int)(ci / ((int64_t)nx * ny));
        double hx = 0, hy = 0, hz = 0;
        for (int kk = 0; kk < nz; ++kk)
        for (int jj = 0; jj < ny; ++jj)
        for (int ii = 0; ii < nx; ++ii) {
            int64_t cj = (int64_t)ii + (int64_t)nx * (jj + (int64_t)ny * kk);
            double ax = Mx[cj], ay = My[cj], az = Mz[cj];
            if (ax == 0.0 && ay == 0.0 && az == 0.0) continue;
            int ox = i - ii, oy = j - jj, oz = k - kk;
            double sx = ox < 0 ? -1.0 : 1.0, sy = oy < 0 ? -1.0 : 1.0, sz = oz < 0 ? -1.0 : 1.0;
            int64_t o = ((int64_t)abs(oz) * ny + abs(oy)) * nx + abs(ox);
            double nxx = tab[o], nyy = tab[P + o], nzz = tab[2 * P + o];
            double nxy = sx * sy * tab[3 * P + o], nxz = sx * sz * tab[4 * P + o], nyz = sy * sz * tab[5 * P + o];
            hx -= nxx * ax + nxy * ay + nxz * az;
            hy -= nxy * ax + nyy * ay + nyz * az;
            hz -= nxz * ax + nyz * ay + nzz * az;
        }
        bx[ci] = ORC_MU0 * hx; by[ci] = ORC_MU0 * hy; bz[ci] = ORC_MU0 * hz;
    }
}

/* ------------------------------------------------------------------------------------------ */
/* Serial MMC with the EXACT demagnetising energy change ("a serial MMC algorithm ... the           */
/* demagnetizing field updated after every accepted move", Appendix B / PAPER.md:218).         */
/* Validation mode of the oracle only: cells are visited one after the other in lexicographic order; for a move   */
/* dM = Ms0 dm of cell c the total demag energy E_d = (mu0 V/2) sum_ij M_i N_ij M_j changes by                    */
/*     dE_d = -V dM . B_d(c) + (mu0 V/2) dM . N(0) . dM        (field term with the CURRENT field + self term),   */
/* and after an accepted move the field of every cell is updated, B_d(i) -= mu0 N(r_i - r_c) dM.                   */
/* tab = octant tensor table of orc_demag_tensor; bx,by,bz = B_d of the state on entry, kept current.              */
/* All other energy terms, the trial move, the random numbers and Eq. (5) are those of orc_visit.                  */
/* ------------------------------------------------------------------------------------------ */
/* beta * dE_d of the move dm of cell c with the current field b (tesla) and the self term; see above */
double orc_exact_demag_dF(const orc_problem *p, const double *tab, const double *bx, const double *by, const double *bz,
                          int64_t c, const double dm[3])
{
    const int64_t P = (int64_t)p->nx * p->ny * p->nz;
    const double V = p->dx * p->dy * p->dz;
    double dM[3] = { p->Ms0[c] * dm[0], p->Ms0[c] * dm[1], p->Ms0[c] * dm[2] };
    double field = -V * (dM[0] * bx[c] + dM[1] * by[c] + dM[2] * bz[c]);
    double self = 0.5 * ORC_MU0 * V * (tab[0] * dM[0] * dM[0] + tab[P] * dM[1] * dM[1] + tab[2 * P] * dM[2] * dM[2]);   /* N(0) is diagonal */
    return p->beta[c] * (field + self);
}

int64_t orc_serial_exact_sweep(const orc_problem *p, double *mx, double *my, double *mz, const double *tab,
                               double *bx, double *by, double *bz, uint64_t sweep, int store_fp32, int64_t *trials_out)
{
    const int nx = p->nx, ny = p->ny, nz = p->nz;
    const int64_t P = (int64_t)nx * ny * nz;
    orc_problem q = *p;
    q.bdx = bx; q.bdy = by; q.bdz = bz;
    int64_t accepted = 0, trials = 0;
    for (int k = 0; k < nz; ++k) for (int j = 0; j < ny; ++j) for (int i = 0; i < nx; ++i) {
        int64_t c = orc_idx(p, i, j, k);
        if (!p->active[c]) continue;
        trials++;
        double u[4];
        orc_cell_uniforms(p->seed, sweep, (uint64_t)c, u);
        double m[3] = { mx[c], my[c], mz[c] };
        double dm[3], f, terms[6];
        orc_trial(m, u, p->one_minus_cos_cone, p->sigma[c], dm, &f);
        orc_cell_dF(&q, mx, my, mz, i, j, k, dm, terms);
        terms[4] = orc_exact_demag_dF(p, tab, bx, by, bz, c, dm);
        double dM[3];
        double dF = terms[0] + terms[1] + terms[2] + terms[3] + terms[4] + terms[5];
        if (!(log(u[3]) - 4.0 * log(f) + dF < 0.0)) continue;
        accepted++;
        double a = m[0] + dm[0], b = m[1] + dm[1], d = m[2] + dm[2];
        if (store_fp32) { a = (double)(float)a; b = (double)(float)b; d = (double)(float)d; }
        dM[0] = p->Ms0[c] * (a - m[0]); dM[1] = p->Ms0[c] * (b - m[1]); dM[2] = p->Ms0[c] * (d - m[2]);
        mx[c] = a; my[c] = b; mz[c] = d;
        #pragma omp parallel for schedule(static)
        for (int64_t ci = 0; ci < P; ++ci) {
            int ii = (int)(ci % nx), jj = (int)((ci / nx) % ny), kk = (int)(ci / ((int64_t)nx * ny));
            int ox = ii - i, oy = jj - j, oz = kk - k;
            double sx = ox < 0 ? -1.0 : 1.0, sy = oy < 0 ? -1.0 : 1.0, sz = oz < 0 ? -1.0 : 1.0;
            int64_t o = ((int64_t)abs(oz) * ny + abs(oy)) * nx + abs(ox);
            double nxx = tab[o], nyy = tab[P + o], nzz = tab[2 * P + o];
            double nxy = sx * sy * tab[3 * P + o], nxz = sx * sz * tab[4 * P + o], nyz = sy * sz * tab[5 * P + o];
            bx[ci] -= ORC_MU0 * (nxx * dM[0] + nxy * dM[1] + nxz * dM[2]);
            by[ci] -= ORC_MU0 * (nxy * dM[0] + nyy * dM[1] + nyz * dM[2]);
            bz[ci] -= ORC_MU0 * (nxz * dM[0] + nyz * dM[1] + nzz * dM[2]);
        }
    }
    if (trials_out) *trials_out = trials;
    return accepted;
}

/*
 * Parity plumbing (stage 2): O4 evaluated for every active cell of one colour with trial
 * vectors supplied by the caller (dm_in[3c+a]) instead of O3's own, so that the energy arithmetic of another
 * implementation can be judged separately from its trigonometry.  No new arithmetic: calls orc_cell_dF.
 */
void orc_colour_terms_given_dm(const orc_problem *p, const double *mx, const double *my, const double *mz,
                               int colour, const double *dm_in, double *terms_out)
{
    #pragma omp parallel for collapse(2) schedule(static)
    for (int k = 0; k < p->nz; ++k)
        for (int j = 0; j < p->ny; ++j)
            for (int i = (j + k + colour) & 1; i < p->nx; i += 2) {
                int64_t c = orc_idx(p, i, j, k);
                if (!p->active[c]) continue;
                orc_cell_dF(p, mx, my, mz, i, j, k, dm_in + 3 * c, terms_out + 6 * c);
            }
}

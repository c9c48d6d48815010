/* dgswem_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT (see dgswem_oracle.h).
 *
 * Plain CPU fp64 oracle of the per-RK-stage hot path of DG-SWEM's explicit time
 * step (arxiv 2508.21208).  It follows the paper's algorithms step by step, in
 * the paper's order: EDGE (Alg. 2) -> GATHER (Alg. 3,
 * PAPER.md:431-457) -> AREA (Alg. 1) -> SSP-RK stage combine
 * -> SLOPELIM -> WETDRY, with WIND at the nodes
 * once per step.  Where the paper is silent the readings of
 * SURVEY.md §8(c) / DESIGN.md "Readings" apply; each is marked [R-n] below.
 *
 * Arithmetic: every expression is written with one IEEE-754 binary64 operation
 * per C operator or fma() call, evaluated left to right as parenthesised.  Sums
 * of products (polynomial evaluation, quadrature accumulation, dot products) are
 * written with the IEEE-754-2008 fusedMultiplyAdd, C99 fma(a,b,c) = a*b+c rounded
 * once, explicitly, where DESIGN.md section 2 says so; the compiler contracts
 * nothing by itself (-ffp-contract=off, no -ffast-math).  The wet/dry decisions
 * are taken in this precision.
 * OpenMP (optional) only parallelises loops whose iterations write disjoint
 * outputs, so the result is bit-identical to the serial run.
 */
#include "dgswem_oracle.h"

#include <math.h>
#include <stdlib.h>
#include <string.h>

/* binary32 build (dgswem_oracle.h): the <math.h> routines called below in their single-precision forms; the tide's
 * sin() stays binary64 (its arguments are) */
#ifdef ORC_F32
#define fma fmaf
#define sqrt sqrtf
#define fabs fabsf
#define rint rintf
#define ldexp ldexpf
#define frexp frexpf
#define ORC_EXP_MAX 80.0f     /* exp arguments beyond +-80 saturate (binary32 range), +-700 in binary64 */
#else
#define ORC_EXP_MAX 700.0
#endif
#ifdef _OPENMP
#include <omp.h>
#endif

/* ------------------------------------------------------------------ basis */
/* Dubiner orthogonal modal basis on the reference triangle (-1,-1),(1,-1),(-1,1),
 * PAPER.md:97-103 eq. (4); mode order 00, 01, 10, then 02, 11, 20, then 03, 12, 21, 30 (p = 3).
 * Input barycentrics; xi_1 = 2 lam_1 - 1, xi_2 = 2 lam_2 - 1.  d1, d2 = d/dxi_1, d/dxi_2.
 * phi_ij = A_i(xi_1, xi_2) B_j^(2i+1)(xi_2) with A_i = P_i(eta_1) s^i (Legendre in the collapsed coordinate, s = (1 - xi_2)/2:
 * A_1 = a = xi_1 + (1 + xi_2)/2, A_2 = (3 a^2 - s^2)/2, A_3 = (5 a^3 - 3 a s^2)/2) and B_j^(alpha) the Jacobi polynomial
 * P_j^(alpha,0): B_1^(3) = (5 y + 3)/2, B_1^(5) = (7 y + 5)/2, B_2^(1) = (5 y^2 + 2 y - 1)/2, B_2^(3) = (21 y^2 + 18 y + 1)/4,
 * B_3^(1) = (35 y^3 + 15 y^2 - 15 y - 3)/8.  All ten modes are always written (callers use the first ndof). */
void orc_basis(real lam0, real lam1, real lam2, real* phi, real* d1, real* d2) {
  (void)lam0;
  real xi1 = RL(2.0) * lam1 - RL(1.0);
  real xi2 = RL(2.0) * lam2 - RL(1.0);
  real s = RL(0.5) * (RL(1.0) - xi2);
  real r = RL(0.5) * (RL(5.0) * xi2 + RL(3.0));
  phi[0] = RL(1.0);
  phi[1] = RL(0.5) * (RL(3.0) * xi2 + RL(1.0));
  phi[2] = xi1 + RL(0.5) * (RL(1.0) + xi2);
  phi[3] = RL(0.5) * (((RL(5.0) * xi2) * xi2 + RL(2.0) * xi2) - RL(1.0));
  phi[4] = phi[2] * r;
  phi[5] = RL(0.5) * ((RL(3.0) * phi[2]) * phi[2] - s * s);
  d1[0] = RL(0.0);            d2[0] = RL(0.0);
  d1[1] = RL(0.0);            d2[1] = RL(1.5);
  d1[2] = RL(1.0);            d2[2] = RL(0.5);
  d1[3] = RL(0.0);            d2[3] = RL(5.0) * xi2 + RL(1.0);
  d1[4] = r;              d2[4] = RL(0.5) * r + RL(2.5) * phi[2];
  d1[5] = RL(3.0) * phi[2];   d2[5] = RL(0.5) * (RL(3.0) * phi[2] + s);
  /* p = 3 */
  {
    const real y = xi2, a = phi[2];
    const real b3 = RL(0.125) * ((((RL(35.0) * y) * y) * y + (RL(15.0) * y) * y) - RL(15.0) * y - RL(3.0));
    const real db3 = RL(0.125) * (((RL(105.0) * y) * y + RL(30.0) * y) - RL(15.0));
    const real b2 = RL(0.25) * (((RL(21.0) * y) * y + RL(18.0) * y) + RL(1.0));
    const real db2 = RL(0.25) * (RL(42.0) * y + RL(18.0));
    const real b1 = RL(0.5) * (RL(7.0) * y + RL(5.0));
    const real a2 = phi[5];                                   /* A_2 */
    const real da2x = d1[5], da2y = d2[5];
    const real a3 = RL(0.5) * (((RL(5.0) * a) * a) * a - ((RL(3.0) * a) * s) * s);
    const real da3x = RL(0.5) * ((RL(15.0) * a) * a - (RL(3.0) * s) * s);
    const real da3y = RL(0.5) * (((RL(7.5) * a) * a - (RL(1.5) * s) * s) + (RL(3.0) * a) * s);
    phi[6] = b3;          d1[6] = RL(0.0);      d2[6] = db3;
    phi[7] = a * b2;      d1[7] = b2;           d2[7] = RL(0.5) * b2 + a * db2;
    phi[8] = a2 * b1;     d1[8] = da2x * b1;    d2[8] = da2y * b1 + RL(3.5) * a2;
    phi[9] = a3;          d1[9] = da3x;         d2[9] = da3y;
  }
}

/* Quadrature [R-5] (paper: "Gauss-Lobatto", no orders): edges Gauss-Legendre
 * with p+1 points; area: p=1 three interior points (2/3,1/6,1/6), p=2 six-point degree-4 rule, p=3 the classical
 * twelve-point degree-6 rule (two 3-point orbits, one 6-point orbit).
 * Reference mass M_ij = 2/((2i+1)(i+j+1)) (diagonal). */
int orc_make_tables(int p, orc_tables* T) {
  memset(T, 0, sizeof(*T));
  if (p != 1 && p != 2 && p != 3) return -1;
  T->p = p;
  T->ndof = (p + 1) * (p + 2) / 2;
  T->nqe = p + 1;
  if (p == 1) {
    T->ge[0] = -RL(0.57735026918962576); T->ge[1] = RL(0.57735026918962576);
    T->we[0] = RL(1.0); T->we[1] = RL(1.0);
    T->nqa = 3;
    for (int i = 0; i < 3; ++i) {
      for (int v = 0; v < 3; ++v) T->la[i][v] = (v == i) ? RL(2.0) / RL(3.0) : RL(1.0) / RL(6.0);
      T->wa[i] = RL(2.0) / RL(3.0);
    }
  } else if (p == 3) {
    T->ge[0] = -RL(0.86113631159405258); T->ge[1] = -RL(0.33998104358485626); T->ge[2] = RL(0.33998104358485626); T->ge[3] = RL(0.86113631159405258);
    T->we[0] = RL(0.34785484513745386); T->we[1] = RL(0.65214515486254614); T->we[2] = RL(0.65214515486254614); T->we[3] = RL(0.34785484513745386);
    T->nqa = 12;
    const real a1 = RL(0.249286745170910), w1 = RL(0.116786275726379);
    const real a2 = RL(0.063089014491502), w2 = RL(0.050844906370207);
    const real b3 = RL(0.053145049844817), c3 = RL(0.310352451033784), w3 = RL(0.082851075618374);
    for (int i = 0; i < 3; ++i) {
      for (int v = 0; v < 3; ++v) {
        T->la[i][v]     = (v == i) ? RL(1.0) - RL(2.0) * a1 : a1;
        T->la[3 + i][v] = (v == i) ? RL(1.0) - RL(2.0) * a2 : a2;
      }
      T->wa[i] = RL(2.0) * w1;
      T->wa[3 + i] = RL(2.0) * w2;
    }
    /* the six permutations of (b3, c3, 1 - b3 - c3) */
    static const int perm[6][3] = {{0, 1, 2}, {0, 2, 1}, {1, 0, 2}, {1, 2, 0}, {2, 0, 1}, {2, 1, 0}};
    const real tri3[3] = {b3, c3, (RL(1.0) - b3) - c3};
    for (int q = 0; q < 6; ++q) {
      for (int v = 0; v < 3; ++v) T->la[6 + q][v] = tri3[perm[q][v]];
      T->wa[6 + q] = RL(2.0) * w3;
    }
  } else {
    T->ge[0] = -RL(0.77459666924148338); T->ge[1] = RL(0.0); T->ge[2] = RL(0.77459666924148338);
    T->we[0] = RL(5.0) / RL(9.0); T->we[1] = RL(8.0) / RL(9.0); T->we[2] = RL(5.0) / RL(9.0);
    T->nqa = 6;
    const real a1 = RL(0.445948490915965), w1 = RL(0.223381589678011);
    const real a2 = RL(0.091576213509771), w2 = RL(0.109951743655322);
    for (int i = 0; i < 3; ++i) {
      for (int v = 0; v < 3; ++v) {
        T->la[i][v]     = (v == i) ? RL(1.0) - RL(2.0) * a1 : a1;
        T->la[3 + i][v] = (v == i) ? RL(1.0) - RL(2.0) * a2 : a2;
      }
      T->wa[i] = RL(2.0) * w1;
      T->wa[3 + i] = RL(2.0) * w2;
    }
  }
  const real M[10] = {RL(2.0), RL(1.0), RL(1.0) / RL(3.0), RL(2.0) / RL(3.0), RL(2.0) / RL(9.0), RL(2.0) / RL(15.0),
                      RL(0.5), RL(1.0) / RL(6.0), RL(0.1), RL(1.0) / RL(14.0)};
  for (int k = 0; k < T->ndof; ++k) T->invM[k] = RL(1.0) / M[k];
  real phi[ORC_MAXDOF], d1[ORC_MAXDOF], d2[ORC_MAXDOF];
  for (int i = 0; i < T->nqa; ++i) {
    orc_basis(T->la[i][0], T->la[i][1], T->la[i][2], phi, d1, d2);
    for (int k = 0; k < T->ndof; ++k) {
      T->phiA[i][k] = phi[k]; T->dphiA1[i][k] = d1[k]; T->dphiA2[i][k] = d2[k];
      T->wfac[i][k] = T->wa[i] * T->invM[k];
      T->srfac[i][k] = T->wfac[i][k] * phi[k];
    }
  }
  for (int j = 0; j < T->nqe; ++j) {
    T->elam[j][0] = RL(0.5) * (RL(1.0) - T->ge[j]);
    T->elam[j][1] = RL(0.5) * (RL(1.0) + T->ge[j]);
  }
  /* local edge l runs from local vertex a=(l+1)%3 to b=(l+2)%3 */
  for (int l = 0; l < 3; ++l) {
    int a = (l + 1) % 3, b = (l + 2) % 3;
    for (int j = 0; j < T->nqe; ++j) {
      real lam[3] = {RL(0.0), RL(0.0), RL(0.0)};
      lam[a] = T->elam[j][0]; lam[b] = T->elam[j][1];
      orc_basis(lam[0], lam[1], lam[2], phi, d1, d2);
      for (int k = 0; k < T->ndof; ++k) {
        T->phiE[l][j][k] = phi[k];
        T->efac[l][j][k] = (T->we[j] * T->invM[k]) * phi[k];
      }
    }
  }
  for (int v = 0; v < 3; ++v) {
    real lam[3] = {RL(0.0), RL(0.0), RL(0.0)};
    lam[v] = RL(1.0);
    orc_basis(lam[0], lam[1], lam[2], phi, d1, d2);
    for (int k = 0; k < T->ndof; ++k) T->phiV[v][k] = phi[k];
  }
  return 0;
}

/* ---------------------------------------------------------- numerical flux */
/* Local Lax-Friedrichs normal flux [R-3] ("e.g., Local Lax-Friedrichs or Roe"),
 * evaluated in the edge frame (n, t), t = (-ny, nx); n points from e+ to e-.
 * Physical flux: eqs (7)-(9) with P = g/2 (H^2 - h_b^2) = g zeta (zeta/2 + h_b).
 * bc: 0 interior, 1 land/wall (mirror: zeta-=zeta+, Qn-=-Qn+, Qt-=Qt+ => mass flux exactly 0),
 *     2 ocean (zeta- = zeta_b, Q- = Q+)   [R-4] (PAPER.md:67 names the boundary types only).
 * Depth floor H_c = max(H, H0) in every denominator and square root [R-6]. */
void orc_llf_flux(real g, real h0, real nx, real ny, real hq,
                  real zp, real qxp, real qyp, real zm, real qxm, real qym,
                  int bc, real zeta_b, real* fz, real* fqx, real* fqy) {
  real qnp = fma(qyp, ny, qxp * nx);
  real qtp = fma(qyp, nx, -(qxp * ny));
  real qnm, qtm;
  if (bc == 0) {
    qnm = fma(qym, ny, qxm * nx);
    qtm = fma(qym, nx, -(qxm * ny));
  } else if (bc == 1) {
    zm = zp; qnm = -qnp; qtm = qtp;
  } else {
    zm = zeta_b; qnm = qnp; qtm = qtp;
  }
  real Hp = zp + hq, Hm = zm + hq;
  real Hcp = (Hp > h0) ? Hp : h0;
  real Hcm = (Hm > h0) ? Hm : h0;
  real rHp = RL(1.0) / Hcp, rHm = RL(1.0) / Hcm;
  real unp = qnp * rHp, unm = qnm * rHm;
  real cp = sqrt(g * Hcp), cm = sqrt(g * Hcm);
  real lp = fabs(unp) + cp, lm = fabs(unm) + cm;
  real lam = (lp > lm) ? lp : lm;
  real hl = RL(0.5) * lam;
  real Pp = (g * zp) * fma(RL(0.5), zp, hq);
  real Pm = (g * zm) * fma(RL(0.5), zm, hq);
  /* each bracket is symmetric in (+,-), so swapping the sides and negating n negates the flux bit for bit */
  real f0 = fma(-hl, zm - zp, RL(0.5) * (qnp + qnm));
  real fn = fma(-hl, qnm - qnp, RL(0.5) * (fma(qnp, unp, Pp) + fma(qnm, unm, Pm)));
  real ft = fma(-hl, qtm - qtp, RL(0.5) * (qtp * unp + qtm * unm));
  *fz = f0;
  *fqx = fma(fn, nx, -(ft * ny));
  *fqy = fma(fn, ny, ft * nx);
}

/* Roe flux [R-17] ("e.g., Local Lax-Friedrichs or Roe"), same frame, boundary states and depth floor as the
 * LLF flux above.  Roe state of the two traces: un~ = (s+ un+ + s- un-)/(s+ + s-), ut~ likewise, s = sqrt(H_c),
 * c~ = sqrt(g (H_c+ + H_c-)/2); jumps dH = zeta- - zeta+ (same bed on both sides), dqn, dqt; wave strengths
 * a1,3 = (dH -+ (dqn - un~ dH)/c~)/2 on lambda1,3 = un~ -+ c~ with r1,3 = (1, lambda1,3, ut~), a2 = dqt - ut~ dH on
 * lambda2 = un~ with r2 = (0, 0, 1);  F^ = (F(w+) + F(w-))/2 . n - (1/2) sum_k |lambda_k| a_k r_k.  No entropy fix.
 * Every two-term sum pairs a "+"-side with a "-"-side product (or wave 1 with wave 3) and is written without fma, so
 * that swapping the sides and negating n negates the flux bit for bit (as for LLF), and a wall has exactly zero mass flux. */
void orc_roe_flux(real g, real h0, real nx, real ny, real hq,
                  real zp, real qxp, real qyp, real zm, real qxm, real qym,
                  int bc, real zeta_b, real* fz, real* fqx, real* fqy) {
  real qnp = fma(qyp, ny, qxp * nx);
  real qtp = fma(qyp, nx, -(qxp * ny));
  real qnm, qtm;
  if (bc == 0) {
    qnm = fma(qym, ny, qxm * nx);
    qtm = fma(qym, nx, -(qxm * ny));
  } else if (bc == 1) {
    zm = zp; qnm = -qnp; qtm = qtp;
  } else {
    zm = zeta_b; qnm = qnp; qtm = qtp;
  }
  real Hp = zp + hq, Hm = zm + hq;
  real Hcp = (Hp > h0) ? Hp : h0;
  real Hcm = (Hm > h0) ? Hm : h0;
  real rHp = RL(1.0) / Hcp, rHm = RL(1.0) / Hcm;
  real unp = qnp * rHp, unm = qnm * rHm;
  real utp = qtp * rHp, utm = qtm * rHm;
  real sp = sqrt(Hcp), sm = sqrt(Hcm);
  real rS = RL(1.0) / (sp + sm);
  real un = (sp * unp + sm * unm) * rS;
  real ut = (sp * utp + sm * utm) * rS;
  real ct = sqrt(g * (RL(0.5) * (Hcp + Hcm)));
  real rc = RL(1.0) / ct;
  real dH = zm - zp, dqn = qnm - qnp, dqt = qtm - qtp;
  real y = (dqn - un * dH) * rc;
  real a1 = RL(0.5) * (dH - y), a3 = RL(0.5) * (dH + y);
  real a2 = dqt - ut * dH;
  real l1 = un - ct, l3 = un + ct;
  real p1 = fabs(l1) * a1, p3 = fabs(l3) * a3;
  real D0 = p1 + p3;
  real Dn = p1 * l1 + p3 * l3;
  real Dt = fma(fabs(un), a2, D0 * ut);
  real Pp = (g * zp) * fma(RL(0.5), zp, hq);
  real Pm = (g * zm) * fma(RL(0.5), zm, hq);
  real f0 = RL(0.5) * ((qnp + qnm) - D0);
  real fn = RL(0.5) * ((fma(qnp, unp, Pp) + fma(qnm, unm, Pm)) - Dn);
  real ft = RL(0.5) * ((qtp * unp + qtm * unm) - Dt);
  *fz = f0;
  *fqx = fma(fn, nx, -(ft * ny));
  *fqy = fma(fn, ny, ft * nx);
}

/* ------------------------------------------------- deterministic exp / log */
/* Used only by the Holland wind: the same short algorithm is implemented independently
 * on the CUDA side so that the nodal wind stress is bit-identical.  Accuracy
 * ~1e-15 relative (pinned against libm in the tests). */
static const real LN2_HI = RL(6.93147180369123816490e-01);
static const real LN2_LO = RL(1.90821492927058770002e-10);
static const real INV_LN2 = RL(1.44269504088896338700e+00);

real orc_det_exp(real x) {
  if (x < -ORC_EXP_MAX) return RL(0.0);
  if (x > ORC_EXP_MAX) x = ORC_EXP_MAX;
  real kf = rint(x * INV_LN2);
  real r = fma(-kf, LN2_LO, fma(-kf, LN2_HI, x));
  /* Taylor series of e^r, |r| <= 0.35, degree 13, Horner */
  real q = RL(1.0) / RL(6227020800.0);
  q = fma(q, r, RL(1.0) / RL(479001600.0));
  q = fma(q, r, RL(1.0) / RL(39916800.0));
  q = fma(q, r, RL(1.0) / RL(3628800.0));
  q = fma(q, r, RL(1.0) / RL(362880.0));
  q = fma(q, r, RL(1.0) / RL(40320.0));
  q = fma(q, r, RL(1.0) / RL(5040.0));
  q = fma(q, r, RL(1.0) / RL(720.0));
  q = fma(q, r, RL(1.0) / RL(120.0));
  q = fma(q, r, RL(1.0) / RL(24.0));
  q = fma(q, r, RL(1.0) / RL(6.0));
  q = fma(q, r, RL(0.5));
  q = fma(q, r, RL(1.0));
  q = fma(q, r, RL(1.0));
  return ldexp(q, (int)kf);
}

real orc_det_log(real x) {
  /* x > 0, finite, normal.  x = m 2^e, m in [sqrt(1/2), sqrt(2)); log m = 2 atanh(s), s=(m-1)/(m+1) */
  int e;
  real m = frexp(x, &e);                 /* m in [0.5, 1) */
  if (m < RL(0.70710678118654752)) { m = RL(2.0) * m; e = e - 1; }
  real f = m - RL(1.0);
  real s = f / (RL(2.0) + f);
  real z = s * s;
  real q = RL(1.0) / RL(23.0);
  q = fma(q, z, RL(1.0) / RL(21.0));
  q = fma(q, z, RL(1.0) / RL(19.0));
  q = fma(q, z, RL(1.0) / RL(17.0));
  q = fma(q, z, RL(1.0) / RL(15.0));
  q = fma(q, z, RL(1.0) / RL(13.0));
  q = fma(q, z, RL(1.0) / RL(11.0));
  q = fma(q, z, RL(1.0) / RL(9.0));
  q = fma(q, z, RL(1.0) / RL(7.0));
  q = fma(q, z, RL(1.0) / RL(5.0));
  q = fma(q, z, RL(1.0) / RL(3.0));
  q = fma(q, z, RL(1.0));
  real ef = (real)e;
  return fma(ef, LN2_LO, fma(ef, LN2_HI, (RL(2.0) * s) * q));
}

/* ------------------------------------------------------------------- wind */
/* WIND (node loops).  [R-9]: analytic Holland (1980) gradient wind about the
 * centre (cx, cy), counter-clockwise; Garratt drag; returns kinematic stress tau_s/rho_0. */
void orc_holland_node(const orc_holland* h, double cx, double cy, real x, real y,
                      real* tsx, real* tsy, real* Vout) {
  orc_holland_node_p(h, RL(0.0), cx, cy, x, y, tsx, tsy, Vout, NULL);
}

/* The same with the Holland (1980) surface pressure p(r) = p_c + dp exp(-(R/r)^B): returns in *etap the pressure
 * anomaly against the far field as a water column, eta_p = (p - p_n)/(rho_0 g) = -(dp/(rho_0 g)) (1 - exp(-(R/r)^B))
 * (PAPER.md:65 forcings, :326 "Wind forcing and pressure calculations (WIND)"; [R-15]).  etap may be NULL. */
void orc_holland_node_p(const orc_holland* h, real g, double cx, double cy, real x, real y,
                        real* tsx, real* tsy, real* Vout, real* etap) {
  /* the vortex parameters arrive as binary64 (API) and are rounded to the working precision once, here */
  const real hB = (real)h->B, hrmax = (real)h->rmax, hdp = (real)h->dp, hra = (real)h->rho_air, hrw = (real)h->rho_water, hf = (real)h->f;
  real dx = x - (real)cx, dy = y - (real)cy;
  real r = sqrt(fma(dy, dy, dx * dx));
  if (r < RL(1.0)) {
    *tsx = RL(0.0); *tsy = RL(0.0); if (Vout) *Vout = RL(0.0);
    if (etap) *etap = -(hdp / (hrw * g));
    return;
  }
  real xb = orc_det_exp(hB * orc_det_log(hrmax / r));   /* (R/r)^B */
  real ee = orc_det_exp(-xb);
  real rf2 = RL(0.5) * (r * hf);
  real V = sqrt(fma((hB / hra) * xb, hdp * ee, rf2 * rf2)) - rf2;
  real rr = RL(1.0) / r;
  real wx = (-(dy * rr)) * V;
  real wy = (dx * rr) * V;
  real cd = fma(RL(0.067), V, RL(0.75)) * RL(1.0e-3);
  if (cd > RL(0.0035)) cd = RL(0.0035);
  real k = ((hra / hrw) * cd) * V;
  *tsx = k * wx;
  *tsy = k * wy;
  if (Vout) *Vout = V;
  if (etap) *etap = -((hdp / (hrw * g)) * (RL(1.0) - ee));
}

/* ---------------------------------------------------------------- limiter */
/* SLOPELIM (PAPER.md:109, :326 -- no algorithm given) [R-7]: edge-neighbour Barth-Jespersen
 * on the linear part of one variable.  w[0]=mean; returns alpha in [0,1]. */
real orc_limit_var(int p, real* w, const real* mean_nb, const int* has_nb) {
  real ubar = w[0];
  real umin = ubar, umax = ubar;
  for (int l = 0; l < 3; ++l) {
    if (!has_nb[l]) continue;
    real m = mean_nb[l];
    if (m < umin) umin = m;
    if (m > umax) umax = m;
  }
  real b = w[1], c = w[2];
  real d[3];
  d[0] = (-b) - c;
  d[1] = (-b) + c;
  d[2] = RL(2.0) * b;
  real alpha = RL(1.0);
  for (int v = 0; v < 3; ++v) {
    real a;
    if (d[v] > RL(0.0)) a = (umax - ubar) / d[v];
    else if (d[v] < RL(0.0)) a = (umin - ubar) / d[v];
    else a = RL(1.0);
    if (a < alpha) alpha = a;
  }
  w[1] = alpha * b;
  w[2] = alpha * c;
  if (p >= 2 && alpha < RL(1.0)) { for (int k = 3; k < (p + 1) * (p + 2) / 2; ++k) w[k] = RL(0.0); }
  return alpha;
}

/* Vertex-neighbourhood Barth-Jespersen (the linearity-preserving variant, SURVEY.md 8(c.2) "known weakness" / 8(f)
 * NEXT-3) [R-18]: the value at vertex v is bounded by the extrema of the means of ALL elements that share that vertex
 * (vmin[v], vmax[v], the element itself included), not by the three edge neighbours.  Same quotient rule and same
 * treatment of the quadratic modes as orc_limit_var. */
real orc_limit_var_vertex(int p, real* w, const real* vmin, const real* vmax) {
  real ubar = w[0];
  real b = w[1], c = w[2];
  real d[3];
  d[0] = (-b) - c;
  d[1] = (-b) + c;
  d[2] = RL(2.0) * b;
  real alpha = RL(1.0);
  for (int v = 0; v < 3; ++v) {
    real a;
    if (d[v] > RL(0.0)) a = (vmax[v] - ubar) / d[v];
    else if (d[v] < RL(0.0)) a = (vmin[v] - ubar) / d[v];
    else a = RL(1.0);
    if (a < alpha) alpha = a;
  }
  w[1] = alpha * b;
  w[2] = alpha * c;
  if (p >= 2 && alpha < RL(1.0)) { for (int k = 3; k < (p + 1) * (p + 2) / 2; ++k) w[k] = RL(0.0); }
  return alpha;
}

/* ---------------------------------------------------------------- wet/dry */
static void vertex_values(const real* w, real* u) {
  /* u(v) = w0 + w1 phi01(v) + w2 phi10(v), phi01 = (-1,-1,2), phi10 = (-1,1,0) */
  real amb = w[0] - w[1];
  u[0] = amb - w[2];
  u[1] = amb + w[2];
  u[2] = fma(RL(2.0), w[1], w[0]);
}
static void modes_from_vertices(const real* u, real* w) {
  real a = ((u[0] + u[1]) + u[2]) / RL(3.0);
  w[0] = a;
  w[1] = RL(0.5) * (u[2] - a);
  w[2] = RL(0.5) * (u[1] - u[0]);
}

/* thin-layer momentum re-assignment (part of [R-8]): vertex weights
 * w_v = clamp((Hh_v - H0)/(H1 - H0), 0, 1), H1 = 10 H0.  Each vertex keeps w_v Q_v; the
 * removed momentum R = sum_v (Q_v - w_v Q_v) is handed back in proportion to w_v, so the
 * element total is conserved (unless every w_v = 0: the momentum is dropped).  Identity when
 * every vertex is deeper than H1. */
static void thin_layer_momentum(real h0, const real* Hh, real* qx, real* qy) {
  const real h1 = RL(10.0) * h0;
  const real rden = RL(1.0) / (h1 - h0);
  real wv[3], W = RL(0.0);
  int all_one = 1;
  for (int v = 0; v < 3; ++v) {
    if (Hh[v] <= h0) wv[v] = RL(0.0);
    else if (Hh[v] >= h1) wv[v] = RL(1.0);
    else wv[v] = (Hh[v] - h0) * rden;
    if (wv[v] != RL(1.0)) all_one = 0;
    W = W + wv[v];
  }
  if (all_one) return;
  real* qq[2] = {qx, qy};
  for (int c = 0; c < 2; ++c) {
    real qv[3], kept[3];
    vertex_values(qq[c], qv);
    real R = RL(0.0);
    for (int v = 0; v < 3; ++v) { kept[v] = wv[v] * qv[v]; R = R + (qv[v] - kept[v]); }
    if (W > RL(0.0)) {
      real share = R / W;
      for (int v = 0; v < 3; ++v) qv[v] = fma(share, wv[v], kept[v]);
    } else {
      for (int v = 0; v < 3; ++v) qv[v] = RL(0.0);
    }
    modes_from_vertices(qv, qq[c]);
  }
}

/* WETDRY (PAPER.md:320, :326 -- no algorithm given) [R-8]: element-local vertex
 * redistribution, SURVEY.md §8(c.3) with the momentum rule replaced by thin_layer_momentum
 * (the survey's equal-share rule pumps momentum into vertices that are
 * barely deeper than H0 and the C4 workload goes non-finite). */
int orc_wetdry_elem(const orc_tables* T, real h0, const real* hv, real* ze, real* qx, real* qy) {
  const int ndof = T->ndof;
  if (T->p >= 2) {
    /* pre-step: full polynomial depth at the vertices, all edge points, all area points;
     * threshold H1 = 10 H0 so that the linear part below governs every thin element */
    const real h1 = RL(10.0) * h0;
    int low = 0;
    for (int v = 0; v < 3 && !low; ++v) {
      real z = ze[0];
      for (int k = 1; k < ndof; ++k) z = fma(ze[k], T->phiV[v][k], z);
      if (z + hv[v] <= h1) low = 1;
    }
    for (int l = 0; l < 3 && !low; ++l) {
      int a = (l + 1) % 3, b = (l + 2) % 3;
      for (int j = 0; j < T->nqe && !low; ++j) {
        real z = ze[0];
        for (int k = 1; k < ndof; ++k) z = fma(ze[k], T->phiE[l][j][k], z);
        real hq = hv[a] * T->elam[j][0] + hv[b] * T->elam[j][1];
        if (z + hq <= h1) low = 1;
      }
    }
    for (int i = 0; i < T->nqa && !low; ++i) {
      real z = ze[0];
      for (int k = 1; k < ndof; ++k) z = fma(ze[k], T->phiA[i][k], z);
      real hq = fma(hv[2], T->la[i][2], fma(hv[1], T->la[i][1], hv[0] * T->la[i][0]));
      if (z + hq <= h1) low = 1;
    }
    if (low) for (int k = 3; k < ndof; ++k) { ze[k] = RL(0.0); qx[k] = RL(0.0); qy[k] = RL(0.0); }
  }
  real zv[3], H[3];
  vertex_values(ze, zv);
  for (int v = 0; v < 3; ++v) H[v] = zv[v] + hv[v];
  if (H[0] > h0 && H[1] > h0 && H[2] > h0) {                     /* (2) no dry vertex: depths untouched */
    thin_layer_momentum(h0, H, qx, qy);
    return 1;
  }
  real Hbar = ((H[0] + H[1]) + H[2]) / RL(3.0);
  real u[3];
  if (Hbar <= h0) {                                               /* (3) dry element */
    for (int v = 0; v < 3; ++v) u[v] = Hbar - hv[v];
    modes_from_vertices(u, ze);
    qx[0] = RL(0.0); qx[1] = RL(0.0); qx[2] = RL(0.0);
    qy[0] = RL(0.0); qy[1] = RL(0.0); qy[2] = RL(0.0);
    return 0;
  }
  /* (4) partially wet: stable ascending sort of the three vertices by H (ties by index) */
  int i1 = 0, i2 = 1, i3 = 2, tmp;
  if (H[i2] < H[i1]) { tmp = i1; i1 = i2; i2 = tmp; }
  if (H[i3] < H[i2]) { tmp = i2; i2 = i3; i3 = tmp; }
  if (H[i2] < H[i1]) { tmp = i1; i1 = i2; i2 = tmp; }
  real Hh[3];
  Hh[i1] = h0;
  real D1 = h0 - H[i1];
  real t2 = H[i2] - RL(0.5) * D1;
  Hh[i2] = (t2 > h0) ? t2 : h0;
  real D2 = Hh[i2] - H[i2];
  Hh[i3] = (H[i3] - D1) - D2;
  for (int v = 0; v < 3; ++v) u[v] = Hh[v] - hv[v];
  modes_from_vertices(u, ze);
  thin_layer_momentum(h0, Hh, qx, qy);
  return 1;
}

/* ----------------------------------------------------------------- SSP-RK */
/* Two-register Shu-Osher SSP Runge-Kutta schemes [R-2, R-19] ("an optimized version of the ... SSPRK"
 * whose coefficients the paper does not print; BASELINE configs name SSP-RK2 / RK3).  Every stage has the form
 *   u = w^(s-1) + (beta_s dt) L(w^(s-1), t + c_s dt);   w^(s) = u  (a_s = 0, b_s = 1)  or  a_s w^0 + b_s u.
 * (order, stages):
 *   (2,2)  SSP(2,2):  beta = 1;    w2 = 1/2 w0 + 1/2 u;                  c = (0, 1)
 *   (3,3)  SSP(3,3):  beta = 1;    w2 = 3/4 w0 + 1/4 u; w3 = 1/3 w0 + 2/3 u;  c = (0, 1, 1/2)
 *   (2,s)  optimal s-stage second-order scheme, s = 3, 4:  beta = 1/(s-1);  w_s = 1/s w0 + (s-1)/s u;  c_i = (i-1)/(s-1)
 *   (3,4)  optimal 4-stage third-order scheme:  beta = 1/2;  w3 = 2/3 w0 + 1/3 u;  c = (0, 1/2, 1, 1/2)
 * The many-stage schemes trade one more L evaluation for a time step (s-1) x (second order) or 2 x (third order) as large. */
typedef struct { int ns; real a[4], b[4]; double beta[4], c[4]; } rk_scheme;
static int rk_get(int order, int stages, rk_scheme* k) {
  if (stages == 0) stages = order;
  memset(k, 0, sizeof(*k));
  k->ns = stages;
  for (int s = 0; s < 4; ++s) { k->a[s] = RL(0.0); k->b[s] = RL(1.0); k->beta[s] = 1.0; k->c[s] = 0.0; }
  if (order == 2 && stages == 2) {
    k->a[1] = RL(0.5); k->b[1] = RL(0.5); k->c[1] = 1.0;
  } else if (order == 3 && stages == 3) {
    k->a[1] = RL(0.75); k->b[1] = RL(0.25); k->c[1] = 1.0;
    k->a[2] = RL(1.0) / RL(3.0); k->b[2] = RL(2.0) / RL(3.0); k->c[2] = 0.5;
  } else if (order == 2 && (stages == 3 || stages == 4)) {
    for (int s = 0; s < stages; ++s) { k->beta[s] = 1.0 / (double)(stages - 1); k->c[s] = (double)s / (double)(stages - 1); }
    k->a[stages - 1] = RL(1.0) / (real)stages; k->b[stages - 1] = (real)(stages - 1) / (real)stages;
  } else if (order == 3 && stages == 4) {
    for (int s = 0; s < 4; ++s) k->beta[s] = 0.5;
    k->c[1] = 0.5; k->c[2] = 1.0; k->c[3] = 0.5;
    k->a[2] = RL(2.0) / RL(3.0); k->b[2] = RL(1.0) / RL(3.0);
  } else {
    return -1;
  }
  return 0;
}

int orc_ssprk_step_s(int order, int stages, int64_t n, real* w, real* w0, real* rhs, double t, double dt,
                     orc_rhs_fn rhs_fn, orc_post_fn post_fn, void* ctx) {
  rk_scheme K;
  if (rk_get(order, stages, &K) != 0) return -1;
  memcpy(w0, w, (size_t)n * sizeof(real));
  for (int s = 0; s < K.ns; ++s) {
    rhs_fn(ctx, s, t + K.c[s] * dt, w, rhs);
    const double dts = K.beta[s] * dt;          /* binary64 like t and dt; rounded once where it meets the state */
    const real a = K.a[s], b = K.b[s];
    if (a == RL(0.0) && b == RL(1.0)) {         /* plain stage: no combine (bitwise: not u + 0 w0) */
#pragma omp parallel for schedule(static)
      for (int64_t i = 0; i < n; ++i) w[i] = fma(dts, rhs[i], w[i]);
    } else {
#pragma omp parallel for schedule(static)
      for (int64_t i = 0; i < n; ++i) {
        real u = fma(dts, rhs[i], w[i]);
        w[i] = fma(b, u, a * w0[i]);
      }
    }
    if (post_fn) post_fn(ctx, s, w);
  }
  return 0;
}

int orc_ssprk_step(int order, int64_t n, real* w, real* w0, real* rhs, double t, double dt,
                   orc_rhs_fn rhs_fn, orc_post_fn post_fn, void* ctx) {
  return orc_ssprk_step_s(order, 0, n, w, w0, rhs, t, dt, rhs_fn, post_fn, ctx);
}

/* ------------------------------------------------------------------ model */
struct orc_model {
  orc_params prm;
  orc_tables T;
  int64_t n_nodes, n_elem, n_edge;
  real *xy, *bathy;
  int32_t *tri, *edge_elem, *edge_bc, *elem_edge;
  int8_t* edge_local;
  /* geometry */
  real *area, *jinv /*[4][ne]*/, *lfac /*[3][ne]*/, *hv /*[3][ne]*/;
  real *enx, *eny, *ehb /*[2][nd]*/;
  int32_t* nbr; /*[3][ne]*/
  /* state: w = [3][ndof][ne] contiguous (ze, qx, qy) */
  real *w, *w0, *rhs, *flux /*[3][nqe][nd]*/, *mean /*[3][ne]*/;
  uint8_t* wet;
  double t;                                   /* time, tide and storm track stay binary64 in every build */
  double tide_amp, tide_omega, tide_phase;
  int wind_on;        /* a Holland vortex is set */
  int stress_on;      /* ... its wind stress enters the momentum source (default 1) */
  int press_on;       /* ... its surface-pressure gradient enters the momentum source (default 0) [R-15] */
  orc_holland hol;
  real *nmin, *nmax; /*[3][nn] extrema of the element means around every node (limiter = 2) */
  real* tau;  /*[2][nn]*/
  real* etap; /*[nn] pressure anomaly as a water column */
  real rain;  /* mass source R of eq. (1), m/s, uniform [R-16] */
};

static void* xmalloc(size_t n) { void* p = malloc(n ? n : 1); if (!p) abort(); return p; }
#define NEW(T, n) ((T*)xmalloc(sizeof(T) * (size_t)(n)))

orc_model* orc_create(const orc_params* prm, int64_t n_nodes, const real* xy, const real* bathy,
                      int64_t n_elem, const int32_t* tri, int64_t n_edge, const int32_t* edge_elem,
                      const int8_t* edge_local, const int32_t* edge_bc, const int32_t* elem_edge) {
  orc_model* m = (orc_model*)calloc(1, sizeof(orc_model));
  m->prm = *prm;
  if (orc_make_tables(prm->p, &m->T) != 0) { free(m); return NULL; }
  { rk_scheme K; if (rk_get(prm->rk_order, prm->rk_stages, &K) != 0) { free(m); return NULL; } }
  m->n_nodes = n_nodes; m->n_elem = n_elem; m->n_edge = n_edge;
  m->xy = NEW(real, 2 * n_nodes); memcpy(m->xy, xy, sizeof(real) * 2 * n_nodes);
  m->bathy = NEW(real, n_nodes); memcpy(m->bathy, bathy, sizeof(real) * n_nodes);
  m->tri = NEW(int32_t, 3 * n_elem); memcpy(m->tri, tri, sizeof(int32_t) * 3 * n_elem);
  m->edge_elem = NEW(int32_t, 2 * n_edge); memcpy(m->edge_elem, edge_elem, sizeof(int32_t) * 2 * n_edge);
  m->edge_local = NEW(int8_t, 2 * n_edge); memcpy(m->edge_local, edge_local, 2 * n_edge);
  m->edge_bc = NEW(int32_t, n_edge); memcpy(m->edge_bc, edge_bc, sizeof(int32_t) * n_edge);
  m->elem_edge = NEW(int32_t, 3 * n_elem); memcpy(m->elem_edge, elem_edge, sizeof(int32_t) * 3 * n_elem);
  const int64_t ne = n_elem, nd = n_edge;
  const int ndof = m->T.ndof, nqe = m->T.nqe;
  m->area = NEW(real, ne); m->jinv = NEW(real, 4 * ne); m->lfac = NEW(real, 3 * ne); m->hv = NEW(real, 3 * ne);
  m->enx = NEW(real, nd); m->eny = NEW(real, nd); m->ehb = NEW(real, 2 * nd);
  m->nbr = NEW(int32_t, 3 * ne);
  /* element geometry (SURVEY.md §8(c.1) "Geometry per element") */
  for (int64_t e = 0; e < ne; ++e) {
    const int32_t* t = tri + 3 * e;
    real x0 = xy[2 * t[0]], y0 = xy[2 * t[0] + 1];
    real x1 = xy[2 * t[1]], y1 = xy[2 * t[1] + 1];
    real x2 = xy[2 * t[2]], y2 = xy[2 * t[2] + 1];
    real dx1 = x1 - x0, dy1 = y1 - y0, dx2 = x2 - x0, dy2 = y2 - y0;
    real A = RL(0.5) * (dx1 * dy2 - dx2 * dy1);
    real rA = RL(1.0) / A;
    m->area[e] = A;
    m->jinv[0 * ne + e] = dy2 * rA;       /* d xi1 / dx */
    m->jinv[1 * ne + e] = (-dx2) * rA;    /* d xi1 / dy */
    m->jinv[2 * ne + e] = (-dy1) * rA;    /* d xi2 / dx */
    m->jinv[3 * ne + e] = dx1 * rA;       /* d xi2 / dy */
    for (int l = 0; l < 3; ++l) {
      int a = t[(l + 1) % 3], b = t[(l + 2) % 3];
      real ex = xy[2 * b] - xy[2 * a], ey = xy[2 * b + 1] - xy[2 * a + 1];
      real L = sqrt(ex * ex + ey * ey);
      m->lfac[l * ne + e] = L * rA;
      m->hv[l * ne + e] = bathy[t[l]];
      int32_t d = elem_edge[3 * e + l];
      int32_t ep = edge_elem[2 * d], em = edge_elem[2 * d + 1];
      int plus = (ep == e && edge_local[2 * d] == l);
      m->nbr[l * ne + e] = plus ? em : ep;
    }
  }
  /* edge geometry, from the e+ side: outward normal of e+, endpoint bathymetry */
  for (int64_t d = 0; d < nd; ++d) {
    int32_t ep = edge_elem[2 * d];
    int lp = edge_local[2 * d];
    int a = tri[3 * ep + (lp + 1) % 3], b = tri[3 * ep + (lp + 2) % 3];
    real ex = xy[2 * b] - xy[2 * a], ey = xy[2 * b + 1] - xy[2 * a + 1];
    real L = sqrt(ex * ex + ey * ey);
    real rL = RL(1.0) / L;
    m->enx[d] = ey * rL;
    m->eny[d] = (-ex) * rL;
    m->ehb[0 * nd + d] = bathy[a];
    m->ehb[1 * nd + d] = bathy[b];
  }
  m->w = NEW(real, 3 * ndof * ne); m->w0 = NEW(real, 3 * ndof * ne); m->rhs = NEW(real, 3 * ndof * ne);
  memset(m->w, 0, sizeof(real) * 3 * ndof * ne);
  m->flux = NEW(real, 3 * nqe * nd); memset(m->flux, 0, sizeof(real) * 3 * nqe * nd);
  m->mean = NEW(real, 3 * ne);
  m->wet = NEW(uint8_t, ne); memset(m->wet, 1, ne);
  m->tau = NEW(real, 2 * n_nodes); memset(m->tau, 0, sizeof(real) * 2 * n_nodes);
  m->etap = NEW(real, n_nodes); memset(m->etap, 0, sizeof(real) * n_nodes);
  m->nmin = NEW(real, 3 * n_nodes); m->nmax = NEW(real, 3 * n_nodes);
  m->stress_on = 1; m->press_on = 0; m->rain = RL(0.0);
  m->t = RL(0.0);
  return m;
}

void orc_destroy(orc_model* m) {
  if (!m) return;
  free(m->xy); free(m->bathy); free(m->tri); free(m->edge_elem); free(m->edge_local); free(m->edge_bc);
  free(m->elem_edge); free(m->area); free(m->jinv); free(m->lfac); free(m->hv); free(m->enx); free(m->eny);
  free(m->ehb); free(m->nbr); free(m->w); free(m->w0); free(m->rhs); free(m->flux); free(m->mean);
  free(m->wet); free(m->tau); free(m->etap); free(m->nmin); free(m->nmax); free(m);
}

const orc_tables* orc_get_tables(const orc_model* m) { return &m->T; }

/* A1 EDGE (Alg. 2): per edge, per edge quadrature point, both traces from the
 * modes of e+ / e- with PHI_EDGE (lines 14-23), numerical flux (line 25).  Instead of adding
 * W+- F^ into EDGE_*[e+-, l+-, k] (lines 35-41) the point fluxes are stored per edge and the
 * weights are applied in the gather (north_star: "edge-flux kernel that writes per-edge fluxes
 * to a buffer"); point j is numbered along e+'s local edge, it is point nqe-1-j of e- [R-10]. */
static void edge_flux_all(orc_model* m, const real* w, real zeta_b) {
  const orc_tables* T = &m->T;
  const int64_t ne = m->n_elem, nd = m->n_edge;
  const int ndof = T->ndof, nqe = T->nqe;
  const real* ze = w; const real* qx = w + (int64_t)ndof * ne; const real* qy = w + 2 * (int64_t)ndof * ne;
#pragma omp parallel for schedule(static)
  for (int64_t d = 0; d < nd; ++d) {
    int32_t ep = m->edge_elem[2 * d], em = m->edge_elem[2 * d + 1];
    int lp = m->edge_local[2 * d], lm = m->edge_local[2 * d + 1];
    int bc = m->edge_bc[d];
    real nx = m->enx[d], ny = m->eny[d];
    real hba = m->ehb[d], hbb = m->ehb[nd + d];
    for (int j = 0; j < nqe; ++j) {
      const real* php = T->phiE[lp][j];
      real zp = ze[ep], qxp = qx[ep], qyp = qy[ep];
      for (int k = 1; k < ndof; ++k) {
        zp = fma(ze[k * ne + ep], php[k], zp);
        qxp = fma(qx[k * ne + ep], php[k], qxp);
        qyp = fma(qy[k * ne + ep], php[k], qyp);
      }
      real zm = RL(0.0), qxm = RL(0.0), qym = RL(0.0);
      if (bc == 0) {
        const real* phm = T->phiE[lm][nqe - 1 - j];
        zm = ze[em]; qxm = qx[em]; qym = qy[em];
        for (int k = 1; k < ndof; ++k) {
          zm = fma(ze[k * ne + em], phm[k], zm);
          qxm = fma(qx[k * ne + em], phm[k], qxm);
          qym = fma(qy[k * ne + em], phm[k], qym);
        }
      }
      real hq = hba * T->elam[j][0] + hbb * T->elam[j][1];   /* symmetric in (a,b): same value from either side */
      real fz, fx, fy;
      if (m->prm.flux == 1) orc_roe_flux(m->prm.g, m->prm.h0_dry, nx, ny, hq, zp, qxp, qyp, zm, qxm, qym, bc, zeta_b, &fz, &fx, &fy);
      else orc_llf_flux(m->prm.g, m->prm.h0_dry, nx, ny, hq, zp, qxp, qyp, zm, qxm, qym, bc, zeta_b, &fz, &fx, &fy);
      m->flux[(0 * nqe + j) * nd + d] = fz;
      m->flux[(1 * nqe + j) * nd + d] = fx;
      m->flux[(2 * nqe + j) * nd + d] = fy;
    }
  }
}

/* A2 GATHER (Alg. 3) then A3 AREA (Alg. 1), A4 inverse mass
 * folded into the weights.  rhs_{c,k} =
 *   - sum_l (L_l/A_e) sum_j EDGEFAC[k,j,l] F^_c(l,j) (+ for the e- side)
 *   + sum_i [ XFAC[k,i] F_c,x + YFAC[k,i] F_c,y + SRFAC[k,i] s_c ]      (volume sign + : [R-1]) */
static void elem_rhs_all(orc_model* m, const real* w, real* rhs, real* scale) {
  const orc_tables* T = &m->T;
  const int64_t ne = m->n_elem, nd = m->n_edge;
  const int ndof = T->ndof, nqe = T->nqe, nqa = T->nqa;
  const real g = m->prm.g, h0 = m->prm.h0_dry, cf = m->prm.cf, fc = m->prm.coriolis_f;
  const real* ze = w; const real* qx = w + (int64_t)ndof * ne; const real* qy = w + 2 * (int64_t)ndof * ne;
#pragma omp parallel for schedule(static)
  for (int64_t e = 0; e < ne; ++e) {
    real r[3][ORC_MAXDOF], sc[3][ORC_MAXDOF];
    for (int c = 0; c < 3; ++c) for (int k = 0; k < ndof; ++k) { r[c][k] = RL(0.0); sc[c][k] = RL(0.0); }
    /* ---- GATHER: local edges 0,1,2 in this fixed order (deterministic) ---- */
    for (int l = 0; l < 3; ++l) {
      int32_t d = m->elem_edge[3 * e + l];
      int plus = (m->edge_elem[2 * d] == e && m->edge_local[2 * d] == l);
      real lf = m->lfac[l * ne + e];
      for (int j = 0; j < nqe; ++j) {
        int jj = plus ? j : nqe - 1 - j;
        for (int c = 0; c < 3; ++c) {
          real t = lf * m->flux[(c * nqe + jj) * nd + d];
          for (int k = 0; k < ndof; ++k) {
            if (plus) r[c][k] = fma(-T->efac[l][j][k], t, r[c][k]); else r[c][k] = fma(T->efac[l][j][k], t, r[c][k]);
            sc[c][k] += fabs(T->efac[l][j][k] * t);
          }
        }
      }
    }
    /* ---- AREA ---- */
    real x1x = m->jinv[e], x1y = m->jinv[ne + e], x2x = m->jinv[2 * ne + e], x2y = m->jinv[3 * ne + e];
    real hv0 = m->hv[e], hv1 = m->hv[ne + e], hv2 = m->hv[2 * ne + e];
    real dhx = RL(0.5) * fma(hv2 - hv0, x2x, (hv1 - hv0) * x1x);   /* grad h_b, constant */
    real dhy = RL(0.5) * fma(hv2 - hv0, x2y, (hv1 - hv0) * x1y);
    int wet = m->wet[e];
    const int32_t* tn = m->tri + 3 * e;
    /* gradient of the pressure anomaly eta_p, linear per element from its nodal values (as grad h_b) [R-15] */
    real dpx = RL(0.0), dpy = RL(0.0);
    const int press = wet && m->wind_on && m->press_on;
    if (press) {
      real p0 = m->etap[tn[0]], p1 = m->etap[tn[1]], p2 = m->etap[tn[2]];
      dpx = RL(0.5) * fma(p2 - p0, x2x, (p1 - p0) * x1x);
      dpy = RL(0.5) * fma(p2 - p0, x2y, (p1 - p0) * x1y);
    }
    const real rain = m->rain;
    for (int i = 0; i < nqa; ++i) {
      real z = ze[e], u_qx = qx[e], u_qy = qy[e];
      for (int k = 1; k < ndof; ++k) {                              /* Alg. 1 lines 10-15 */
        z = fma(ze[k * ne + e], T->phiA[i][k], z);
        u_qx = fma(qx[k * ne + e], T->phiA[i][k], u_qx);
        u_qy = fma(qy[k * ne + e], T->phiA[i][k], u_qy);
      }
      real hq = fma(hv2, T->la[i][2], fma(hv1, T->la[i][1], hv0 * T->la[i][0]));
      real H = z + hq;
      real Hc = (H > h0) ? H : h0;
      real rH = RL(1.0) / Hc;
      real u = u_qx * rH, v = u_qy * rH;
      real gz = g * z;
      real P = gz * fma(RL(0.5), z, hq);
      real F[3][2];                                               /* eqs (7)-(9) */
      F[0][0] = u_qx;         F[0][1] = u_qy;
      F[1][0] = fma(u_qx, u, P); F[1][1] = u_qx * v;
      F[2][0] = F[1][1];         F[2][1] = fma(u_qy, v, P);
      real tau = RL(0.0), tsx = RL(0.0), tsy = RL(0.0);
      if (wet) {                                                    /* friction, wind: wet elements only [R-6] */
        tau = (cf * sqrt(fma(u_qy, u_qy, u_qx * u_qx))) * (rH * rH);
        if (m->wind_on && m->stress_on) {
          /* wind stress, linear from the three nodes, ramped by the local depth with the same
           * thin-layer weight as the wet/dry momentum rule: clamp((H-H0)/(H1-H0),0,1), H1=10 H0
           * ([R-9]; a millimetre film must not take the full hurricane stress: tau_s/H is stiff) */
          const real* tx = m->tau; const real* ty = m->tau + m->n_nodes;
          real ramp;
          if (H <= h0) ramp = RL(0.0);
          else if (H >= RL(10.0) * h0) ramp = RL(1.0);
          else ramp = (H - h0) * (RL(1.0) / (RL(10.0) * h0 - h0));
          tsx = ramp * fma(tx[tn[2]], T->la[i][2], fma(tx[tn[1]], T->la[i][1], tx[tn[0]] * T->la[i][0]));
          tsy = ramp * fma(ty[tn[2]], T->la[i][2], fma(ty[tn[1]], T->la[i][1], ty[tn[0]] * T->la[i][0]));
        }
      }
      real S[3];
      S[0] = rain;                                                  /* mass source R of eq. (1) [R-16] */
      S[1] = fma(fc, u_qy, fma(-tau, u_qx, gz * dhx)) + tsx;
      S[2] = fma(-fc, u_qx, fma(-tau, u_qy, gz * dhy)) + tsy;
      real gH = RL(0.0);
      if (press) {                                                  /* -(H/rho_0) grad p_a = -g H grad eta_p [R-15] */
        gH = g * H;
        S[1] = fma(-gH, dpx, S[1]);
        S[2] = fma(-gH, dpy, S[2]);
      }
      for (int k = 0; k < ndof; ++k) {                              /* Alg. 1 lines 26-35 */
        real gxk = fma(T->dphiA2[i][k], x2x, T->dphiA1[i][k] * x1x);
        real gyk = fma(T->dphiA2[i][k], x2y, T->dphiA1[i][k] * x1y);
        real xf = T->wfac[i][k] * gxk, yf = T->wfac[i][k] * gyk, sf = T->srfac[i][k];
        r[0][k] = fma(yf, F[0][1], fma(xf, F[0][0], r[0][k]));
        if (rain != RL(0.0)) r[0][k] = fma(sf, S[0], r[0][k]);
        r[1][k] = fma(sf, S[1], fma(yf, F[1][1], fma(xf, F[1][0], r[1][k])));
        r[2][k] = fma(sf, S[2], fma(yf, F[2][1], fma(xf, F[2][0], r[2][k])));
        for (int c = 0; c < 3; ++c)
          sc[c][k] += fabs(xf * F[c][0]) + fabs(yf * F[c][1]) + (c ? fabs(sf * (gz * (c == 1 ? dhx : dhy))) +
                      fabs(sf * (tau * (c == 1 ? u_qx : u_qy))) + fabs(sf * (fc * (c == 1 ? u_qy : u_qx))) +
                      fabs(sf * (c == 1 ? tsx : tsy)) + fabs(sf * (gH * (c == 1 ? dpx : dpy))) : fabs(sf * S[0]));
      }
    }
    for (int c = 0; c < 3; ++c)
      for (int k = 0; k < ndof; ++k) {
        rhs[((int64_t)c * ndof + k) * ne + e] = r[c][k];
        if (scale) scale[((int64_t)c * ndof + k) * ne + e] = sc[c][k];
      }
  }
}

static double tide_value(const orc_model* m, double t) {
  if (m->tide_amp == 0.0) return 0.0;
  return m->tide_amp * sin(m->tide_omega * t + m->tide_phase);
}

static void dg_rhs(void* ctx, int stage, double t_stage, const real* w, real* rhs) {
  (void)stage;
  orc_model* m = (orc_model*)ctx;
  edge_flux_all(m, w, tide_value(m, t_stage));
  elem_rhs_all(m, w, rhs, NULL);
}

/* A6 SLOPELIM over all elements, then A7 WETDRY over all elements (order RK -> limiter ->
 * wet/dry, [R-7]/[R-8]).  The limiter reads the RK-updated, not yet limited means; it never
 * changes a mean, so the in-place sweep equals the Jacobi sweep.  The wet flag used by the
 * limiter is the one from the end of the previous stage. */
static void limiter_all(orc_model* m, real* w) {
  const int64_t ne = m->n_elem;
  const int ndof = m->T.ndof, p = m->T.p;
#pragma omp parallel for schedule(static)
  for (int64_t e = 0; e < ne; ++e) for (int c = 0; c < 3; ++c) m->mean[c * ne + e] = w[((int64_t)c * ndof) * ne + e];
  if (m->prm.limiter == 2) {
    /* extrema of the means of the elements around every node (every incident element counts, wet or dry);
     * min / max do not depend on the order of the sweep */
    const int64_t nn = m->n_nodes;
    for (int c = 0; c < 3; ++c)
      for (int64_t n = 0; n < nn; ++n) { m->nmin[c * nn + n] = INFINITY; m->nmax[c * nn + n] = -INFINITY; }
    for (int64_t e = 0; e < ne; ++e)
      for (int v = 0; v < 3; ++v) {
        const int64_t n = m->tri[3 * e + v];
        for (int c = 0; c < 3; ++c) {
          const real mu = m->mean[c * ne + e];
          if (mu < m->nmin[c * nn + n]) m->nmin[c * nn + n] = mu;
          if (mu > m->nmax[c * nn + n]) m->nmax[c * nn + n] = mu;
        }
      }
#pragma omp parallel for schedule(static)
    for (int64_t e = 0; e < ne; ++e) {
      if (!m->wet[e]) continue;
      for (int c = 0; c < 3; ++c) {
        real wl[ORC_MAXDOF], lo[3], hi[3];
        for (int k = 0; k < ndof; ++k) wl[k] = w[((int64_t)c * ndof + k) * ne + e];
        for (int v = 0; v < 3; ++v) {
          const int64_t n = m->tri[3 * e + v];
          lo[v] = m->nmin[c * nn + n]; hi[v] = m->nmax[c * nn + n];
        }
        orc_limit_var_vertex(p, wl, lo, hi);
        for (int k = 1; k < ndof; ++k) w[((int64_t)c * ndof + k) * ne + e] = wl[k];
      }
    }
    return;
  }
#pragma omp parallel for schedule(static)
  for (int64_t e = 0; e < ne; ++e) {
    if (!m->wet[e]) continue;
    for (int c = 0; c < 3; ++c) {
      real wl[ORC_MAXDOF], mn[3];
      int has[3];
      for (int k = 0; k < ndof; ++k) wl[k] = w[((int64_t)c * ndof + k) * ne + e];
      for (int l = 0; l < 3; ++l) {
        int32_t nb = m->nbr[l * ne + e];
        has[l] = nb >= 0;
        mn[l] = has[l] ? m->mean[c * ne + nb] : RL(0.0);
      }
      orc_limit_var(p, wl, mn, has);
      for (int k = 1; k < ndof; ++k) w[((int64_t)c * ndof + k) * ne + e] = wl[k];
    }
  }
}

static void wetdry_all(orc_model* m, real* w) {
  const int64_t ne = m->n_elem;
  const int ndof = m->T.ndof;
#pragma omp parallel for schedule(static)
  for (int64_t e = 0; e < ne; ++e) {
    real ze[ORC_MAXDOF], qx[ORC_MAXDOF], qy[ORC_MAXDOF], hv[3];
    for (int k = 0; k < ndof; ++k) {
      ze[k] = w[(0 * (int64_t)ndof + k) * ne + e];
      qx[k] = w[(1 * (int64_t)ndof + k) * ne + e];
      qy[k] = w[(2 * (int64_t)ndof + k) * ne + e];
    }
    for (int v = 0; v < 3; ++v) hv[v] = m->hv[v * ne + e];
    m->wet[e] = (uint8_t)orc_wetdry_elem(&m->T, m->prm.h0_dry, hv, ze, qx, qy);
    for (int k = 0; k < ndof; ++k) {
      w[(0 * (int64_t)ndof + k) * ne + e] = ze[k];
      w[(1 * (int64_t)ndof + k) * ne + e] = qx[k];
      w[(2 * (int64_t)ndof + k) * ne + e] = qy[k];
    }
  }
}

static void dg_post(void* ctx, int stage, real* w) {
  (void)stage;
  orc_model* m = (orc_model*)ctx;
  if (m->prm.limiter) limiter_all(m, w);
  if (m->prm.wetdry) wetdry_all(m, w);
}

/* A0 WIND at t_n, frozen over the stages of the step [R-9] */
static void wind_all(orc_model* m, double t) {
  double cx = m->hol.x0 + m->hol.vx * t, cy = m->hol.y0 + m->hol.vy * t;
  const int64_t nn = m->n_nodes;
#pragma omp parallel for schedule(static)
  for (int64_t i = 0; i < nn; ++i)
    orc_holland_node_p(&m->hol, m->prm.g, cx, cy, m->xy[2 * i], m->xy[2 * i + 1], &m->tau[i], &m->tau[nn + i], NULL, &m->etap[i]);
}

void orc_set_state(orc_model* m, double t, const real* ze, const real* qx, const real* qy) {
  const int64_t n = (int64_t)m->T.ndof * m->n_elem;
  memcpy(m->w, ze, sizeof(real) * n);
  memcpy(m->w + n, qx, sizeof(real) * n);
  memcpy(m->w + 2 * n, qy, sizeof(real) * n);
  m->t = t;
  memset(m->wet, 1, m->n_elem);
  if (m->prm.wetdry) wetdry_all(m, m->w);       /* initialises the wet mask */
}

/* TEST HOOKS for the pins of limiter_all / wetdry_all (no arithmetic of their own): load a state and wet flags as
 * given, without the initial wet/dry pass; apply the post-stage sequence SLOPELIM -> WETDRY (either part optional)
 * to the current state exactly as a stage does. */
void orc_set_state_raw(orc_model* m, double t, const real* ze, const real* qx, const real* qy, const uint8_t* wet) {
  const int64_t n = (int64_t)m->T.ndof * m->n_elem;
  memcpy(m->w, ze, sizeof(real) * n);
  memcpy(m->w + n, qx, sizeof(real) * n);
  memcpy(m->w + 2 * n, qy, sizeof(real) * n);
  m->t = t;
  memcpy(m->wet, wet, (size_t)m->n_elem);
}

void orc_apply_post(orc_model* m, int do_limiter, int do_wetdry) {
  if (do_limiter) limiter_all(m, m->w);
  if (do_wetdry) wetdry_all(m, m->w);
}

void orc_set_tide(orc_model* m, double amp, double omega, double phase) {
  m->tide_amp = amp; m->tide_omega = omega; m->tide_phase = phase;
}

void orc_set_wind_holland(orc_model* m, const orc_holland* h) {
  if (h) { m->hol = *h; m->wind_on = 1; } else { m->wind_on = 0; }
}

/* which parts of the Holland forcing enter the momentum source (defaults: stress on, pressure gradient off) */
void orc_set_wind_forcing(orc_model* m, int stress_on, int press_on) { m->stress_on = stress_on != 0; m->press_on = press_on != 0; }

/* uniform mass source R (rain) in m/s */
void orc_set_rain(orc_model* m, real rate) { m->rain = rate; }

void orc_step(orc_model* m, int64_t nsteps, double dt) {
  const int64_t n = 3 * (int64_t)m->T.ndof * m->n_elem;
  for (int64_t s = 0; s < nsteps; ++s) {
    if (m->wind_on) wind_all(m, m->t);
    orc_ssprk_step_s(m->prm.rk_order, m->prm.rk_stages, n, m->w, m->w0, m->rhs, m->t, dt, dg_rhs, dg_post, m);
    m->t = m->t + dt;
  }
}

void orc_eval_rhs(orc_model* m, real* rze, real* rqx, real* rqy, real* sze, real* sqx, real* sqy) {
  const int64_t n = (int64_t)m->T.ndof * m->n_elem;
  if (m->wind_on) wind_all(m, m->t);
  edge_flux_all(m, m->w, tide_value(m, m->t));
  real* sc = (sze && sqx && sqy) ? NEW(real, 3 * n) : NULL;
  elem_rhs_all(m, m->w, m->rhs, sc);
  memcpy(rze, m->rhs, sizeof(real) * n);
  memcpy(rqx, m->rhs + n, sizeof(real) * n);
  memcpy(rqy, m->rhs + 2 * n, sizeof(real) * n);
  if (sc) {
    memcpy(sze, sc, sizeof(real) * n); memcpy(sqx, sc + n, sizeof(real) * n); memcpy(sqy, sc + 2 * n, sizeof(real) * n);
    free(sc);
  }
}

void orc_get_flux(orc_model* m, real* flux) {
  memcpy(flux, m->flux, sizeof(real) * 3 * (size_t)m->T.nqe * (size_t)m->n_edge);
}

void orc_get_state(orc_model* m, double* t, real* ze, real* qx, real* qy) {
  const int64_t n = (int64_t)m->T.ndof * m->n_elem;
  if (t) *t = m->t;
  memcpy(ze, m->w, sizeof(real) * n);
  memcpy(qx, m->w + n, sizeof(real) * n);
  memcpy(qy, m->w + 2 * n, sizeof(real) * n);
}

/* Nodal output ("to output the state variables, we convert the modal representation to a nodal
 * representation by averaging the neighboring elements of each node"): value of every incident element's polynomial at
 * the node (basis at the vertices, modes k ascending), summed in ascending element order, divided by the count. */
void orc_get_nodal(orc_model* m, real* zn, real* qxn, real* qyn) {
  const int64_t ne = m->n_elem, nn = m->n_nodes;
  const int ndof = m->T.ndof;
  real* out[3] = {zn, qxn, qyn};
  int32_t* cnt = (int32_t*)calloc((size_t)nn, sizeof(int32_t));
  for (int c = 0; c < 3; ++c) for (int64_t n = 0; n < nn; ++n) out[c][n] = RL(0.0);
  for (int64_t e = 0; e < ne; ++e) {
    for (int v = 0; v < 3; ++v) {
      const int64_t n = m->tri[3 * e + v];
      for (int c = 0; c < 3; ++c) {
        const real* w = m->w + ((int64_t)c * ndof) * ne;
        real val = w[e];
        for (int k = 1; k < ndof; ++k) val = fma(w[(int64_t)k * ne + e], m->T.phiV[v][k], val);
        out[c][n] = out[c][n] + val;
      }
      cnt[n] += 1;
    }
  }
  for (int c = 0; c < 3; ++c) for (int64_t n = 0; n < nn; ++n) if (cnt[n] > 0) out[c][n] = out[c][n] / (real)cnt[n];
  free(cnt);
}

void orc_get_wetdry(orc_model* m, uint8_t* wet) { memcpy(wet, m->wet, (size_t)m->n_elem); }

void orc_get_geometry(orc_model* m, real* area, real* jinv, real* lfac, real* enx, real* eny) {
  if (area) memcpy(area, m->area, sizeof(real) * m->n_elem);
  if (jinv) memcpy(jinv, m->jinv, sizeof(real) * 4 * m->n_elem);
  if (lfac) memcpy(lfac, m->lfac, sizeof(real) * 3 * m->n_elem);
  if (enx) memcpy(enx, m->enx, sizeof(real) * m->n_edge);
  if (eny) memcpy(eny, m->eny, sizeof(real) * m->n_edge);
}

void orc_get_wind(orc_model* m, real* tau) { memcpy(tau, m->tau, sizeof(real) * 2 * m->n_nodes); }

void orc_get_pressure(orc_model* m, real* etap) { memcpy(etap, m->etap, sizeof(real) * m->n_nodes); }

int orc_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

/*
 * gprfwi_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, float64 CPU statement of the hot path of arxiv/paper_2506_20513
 * (GPR dual-parameter FWI): the 2-D TM-mode (Ez, Hx, Hy) Yee FDTD in lossy
 * media with CPML, run forward (Algorithm 1) and then as its
 * hand-derived exact discrete adjoint (Algorithm 2) to give
 * d(sum residual*trace)/d(eps_r) and /d(sigma).  The relative permeability mu_r is an optional
 * per-cell model input (Table 1 `miu`; it is not inverted for).
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may build, load or call this file.  It shares no code
 * with paper_2506_20513_b200/csrc and must never be called from the product.
 *
 * The loops follow the paper's order and notation with no blocking, fusion or
 * reordering: one pass per stage of Algorithm 1 / Algorithm 2.  The only
 * concession to run time is "#pragma omp parallel for" over grid rows.
 *
 * The file is compiled twice: once with SCALAR = double (prefix oracle_) and
 * once with -DORACLE_COMPLEX, SCALAR = double _Complex (prefix oraclez_), so
 * that the *same* forward loop gives complex-step directional derivatives
 * (pin 4 in DESIGN.md).  CPML tables, dx, dt and the wavelet stay real.
 *
 * Readings of the paper where it is silent/garbled are DESIGN.md section 3
 * (R1..R14); each is named where it is used.
 *
 * Parity pins (tests/test_oracle_pins.py): analytic 2-D line-source Green's
 * function, discrete energy conservation, reciprocity, adjoint identity via
 * complex step, central finite differences, sigma=0 / PEC / npml=0 special
 * cases, CPML-vs-big-box, linearity and shot independence, checkpointed ==
 * stored history.  No function here is "parity unpinned".
 *
 * Index conventions: full grid NZ x NX Ez nodes incl. CPML;
 * j = z (slow), i = x (fast).  Ez at (j,i); Hx at (j+1/2,i), array (NZ-1) x NX;
 * Hy at (j,i+1/2), array NZ x (NX-1).  eps_r, sigma collocated with Ez.
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#include <stdint.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#ifdef ORACLE_COMPLEX
#include <complex.h>
typedef double _Complex SCALAR;
#define FN(name) oraclez_##name
#define REALPART(x) creal(x)
#else
typedef double SCALAR;
#define FN(name) oracle_##name
#define REALPART(x) (x)
#endif

/* physical constants (paper names them m0, e0 only) */
#define C0   299792458.0
#define PI_  3.14159265358979323846
#define MU0  (4.0e-7 * PI_)
#define EPS0 (1.0 / (MU0 * C0 * C0))

typedef struct {
  int32_t nz, nx;            /* full grid incl. CPML                                  */
  double  dx, dt;            /* square cells (paper uses one uE1 for both directions) */
  int32_t nt;
  int32_t npml, pml_order;   /* CPML thickness P (0 = PEC box) and grading m          */
  double  pml_sigma_max, pml_kappa_max, pml_alpha_max;
  int32_t nshots, nrec;
  int32_t wavelet_per_shot;  /* 0: wavelet[nt] shared; 1: wavelet[nshots][nt]         */
} oracle_params;

/* ---------------------------------------------------------------------------------------
 * Coefficients -- paper's `ucget` kernel, PAPER.md:291-306 (listing truncated after EA;
 * reading R2): EA = e0*er/dt + sigma/2, EB = e0*er/dt - sigma/2, Ca = uE0 = EB/EA,
 * Cb = uE4 = 1/EA.  sigma > 100 S/m => PEC, Ca = Cb = 0.
 * Semi-implicit loss term (reading R1), not Eq. (3)'s explicit one.
 * ------------------------------------------------------------------------------------- */
void FN(coefficients)(int64_t n, const SCALAR *eps_r, const SCALAR *sigma, double dt,
                      SCALAR *Ca, SCALAR *Cb)
{
  for (int64_t k = 0; k < n; ++k) {
    if (REALPART(sigma[k]) > 100.0) { Ca[k] = 0.0; Cb[k] = 0.0; continue; }
    SCALAR EA = EPS0 * eps_r[k] / dt + 0.5 * sigma[k];
    SCALAR EB = EPS0 * eps_r[k] / dt - 0.5 * sigma[k];
    Ca[k] = EB / EA;
    Cb[k] = 1.0 / EA;
  }
}

/* ---------------------------------------------------------------------------------------
 * CPML 1-D profile (reading R4: Roden-Gedney CPML with CFS stretching; the paper only
 * says "two PML kernels").  Axis with N Ez nodes, thickness P.
 * half = 0: E-located table, N entries, position p = i.
 * half = 1: H-located table, N-1 entries, position p = i + 1/2.
 * depth d = max(P - p, p - (N-1-P), 0), rho = d/P;
 * sigma_p = smax*rho^m, kappa = 1 + (kmax-1)*rho^m, alpha = amax*(1-rho);
 * rho > 0: b = exp(-(sigma_p/kappa + alpha)*dt/eps0),
 *          c = sigma_p*(b-1)/(kappa*(sigma_p + kappa*alpha))  (0 if denominator is 0);
 * rho = 0: b = 0, c = 0, kappa = 1.   Output ik = 1/kappa.
 * ------------------------------------------------------------------------------------- */
#ifndef ORACLE_COMPLEX
void oracle_cpml_profile(int N, int P, int m, double smax, double kmax, double amax, double dt,
                         int half, double *b, double *c, double *ik)
{
  int len = half ? N - 1 : N;
  for (int i = 0; i < len; ++i) {
    double p = half ? i + 0.5 : (double)i;
    double d = 0.0;
    if (P > 0) {
      double dl = P - p, dr = p - (N - 1 - P);
      d = dl > dr ? dl : dr;
      if (d < 0.0) d = 0.0;
    }
    if (d <= 0.0) { b[i] = 0.0; c[i] = 0.0; ik[i] = 1.0; continue; }
    double rho = d / P;
    double rm = pow(rho, (double)m);
    double sp = smax * rm;
    double kap = 1.0 + (kmax - 1.0) * rm;
    double al = amax * (1.0 - rho);
    double bb = exp(-(sp / kap + al) * dt / EPS0);
    double den = kap * (sp + kap * al);
    b[i] = bb;
    c[i] = den != 0.0 ? sp * (bb - 1.0) / den : 0.0;
    ik[i] = 1.0 / kap;
  }
}

int oracle_num_threads(void)
{
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}
#else
void oracle_cpml_profile(int N, int P, int m, double smax, double kmax, double amax, double dt,
                         int half, double *b, double *c, double *ik);
#endif

/* all per-shot state of the scheme */
typedef struct {
  int nz, nx;
  SCALAR *Ez;    /* [nz][nx]     */
  SCALAR *Hx;    /* [nz-1][nx]   */
  SCALAR *Hy;    /* [nz][nx-1]   */
  SCALAR *pHxz;  /* [nz-1][nx]   psi of dEz/dz in the Hx update */
  SCALAR *pHyx;  /* [nz][nx-1]   psi of dEz/dx in the Hy update */
  SCALAR *pEzx;  /* [nz][nx]     psi of dHy/dx in the Ez update */
  SCALAR *pEzz;  /* [nz][nx]     psi of dHx/dz in the Ez update */
} state_t;

typedef struct {
  double *b_ex, *c_ex, *ik_ex;   /* [nx]   */
  double *b_ez, *c_ez, *ik_ez;   /* [nz]   */
  double *b_hx, *c_hx, *ik_hx;   /* [nx-1] */
  double *b_hz, *c_hz, *ik_hz;   /* [nz-1] */
} tables_t;

static size_t state_count(int nz, int nx)
{
  return (size_t)nz * nx * 3 + (size_t)(nz - 1) * nx * 2 + (size_t)nz * (nx - 1) * 2;
}

static SCALAR *state_alloc(state_t *s, int nz, int nx)
{
  SCALAR *buf = (SCALAR *)calloc(state_count(nz, nx), sizeof(SCALAR));
  if (!buf) return NULL;
  SCALAR *p = buf;
  s->nz = nz; s->nx = nx;
  s->Ez = p;   p += (size_t)nz * nx;
  s->pEzx = p; p += (size_t)nz * nx;
  s->pEzz = p; p += (size_t)nz * nx;
  s->Hx = p;   p += (size_t)(nz - 1) * nx;
  s->pHxz = p; p += (size_t)(nz - 1) * nx;
  s->Hy = p;   p += (size_t)nz * (nx - 1);
  s->pHyx = p;
  return buf;
}

static int tables_alloc(tables_t *t, const oracle_params *p)
{
  int nz = p->nz, nx = p->nx;
  size_t tot = 3 * ((size_t)nx + nz + (nx - 1) + (nz - 1));
  double *buf = (double *)calloc(tot, sizeof(double));
  if (!buf) return -1;
  double *q = buf;
  t->b_ex = q; q += nx; t->c_ex = q; q += nx; t->ik_ex = q; q += nx;
  t->b_ez = q; q += nz; t->c_ez = q; q += nz; t->ik_ez = q; q += nz;
  t->b_hx = q; q += nx - 1; t->c_hx = q; q += nx - 1; t->ik_hx = q; q += nx - 1;
  t->b_hz = q; q += nz - 1; t->c_hz = q; q += nz - 1; t->ik_hz = q; q += nz - 1;
  oracle_cpml_profile(nx, p->npml, p->pml_order, p->pml_sigma_max, p->pml_kappa_max,
                      p->pml_alpha_max, p->dt, 0, t->b_ex, t->c_ex, t->ik_ex);
  oracle_cpml_profile(nz, p->npml, p->pml_order, p->pml_sigma_max, p->pml_kappa_max,
                      p->pml_alpha_max, p->dt, 0, t->b_ez, t->c_ez, t->ik_ez);
  oracle_cpml_profile(nx, p->npml, p->pml_order, p->pml_sigma_max, p->pml_kappa_max,
                      p->pml_alpha_max, p->dt, 1, t->b_hx, t->c_hx, t->ik_hx);
  oracle_cpml_profile(nz, p->npml, p->pml_order, p->pml_sigma_max, p->pml_kappa_max,
                      p->pml_alpha_max, p->dt, 1, t->b_hz, t->c_hz, t->ik_hz);
  return 0;
}
static void tables_free(tables_t *t) { free(t->b_ex); }

/* ---------------------------------------------------------------------------------------
 * One forward time step n -> n+1 of one shot, stages 2-6 of Algorithm 1.
 * Stage 1 (receivers) and 7 (save wavefield) are done by the caller around this.
 * ------------------------------------------------------------------------------------- */
static void forward_step(state_t *s, const tables_t *t, const SCALAR *Ca, const SCALAR *Cb,
                         double dx, const double *Db, int src_z, int src_x, double w_n)
{
  const int nz = s->nz, nx = s->nx;
  /* stages 2-3: magnetic update + magnetic PML.  Eq. (4) */
#pragma omp parallel for schedule(static)
  for (int j = 0; j <= nz - 2; ++j)
    for (int i = 0; i < nx; ++i) {
      size_t k = (size_t)j * nx + i;
      SCALAR g = (s->Ez[(size_t)(j + 1) * nx + i] - s->Ez[(size_t)j * nx + i]) / dx;
      s->pHxz[k] = t->b_hz[j] * s->pHxz[k] + t->c_hz[j] * g;
      s->Hx[k] -= Db[(size_t)j * nx + i] * (g * t->ik_hz[j] + s->pHxz[k]);
    }
  /* Eq. (5) */
#pragma omp parallel for schedule(static)
  for (int j = 0; j < nz; ++j)
    for (int i = 0; i <= nx - 2; ++i) {
      size_t k = (size_t)j * (nx - 1) + i;
      SCALAR g = (s->Ez[(size_t)j * nx + i + 1] - s->Ez[(size_t)j * nx + i]) / dx;
      s->pHyx[k] = t->b_hx[i] * s->pHyx[k] + t->c_hx[i] * g;
      s->Hy[k] += Db[(size_t)j * nx + i] * (g * t->ik_hx[i] + s->pHyx[k]);
    }
  /* stages 4-5: electric update + electric PML.  Eq. (3) in Ca/Cb form.
   * Outer ring of Ez nodes is PEC and never updated (reading R5). */
#pragma omp parallel for schedule(static)
  for (int j = 1; j <= nz - 2; ++j)
    for (int i = 1; i <= nx - 2; ++i) {
      size_t k = (size_t)j * nx + i;
      SCALAR gx = (s->Hy[(size_t)j * (nx - 1) + i] - s->Hy[(size_t)j * (nx - 1) + i - 1]) / dx;
      SCALAR gz = (s->Hx[(size_t)j * nx + i] - s->Hx[(size_t)(j - 1) * nx + i]) / dx;
      s->pEzx[k] = t->b_ex[i] * s->pEzx[k] + t->c_ex[i] * gx;
      s->pEzz[k] = t->b_ez[j] * s->pEzz[k] + t->c_ez[j] * gz;
      SCALAR K = gx * t->ik_ex[i] + s->pEzx[k] - gz * t->ik_ez[j] - s->pEzz[k];
      s->Ez[k] = Ca[k] * s->Ez[k] + Cb[k] * K;
    }
  /* stage 6: source.  PAPER.md:364-384 with dl = dz (reading R7): Ez -= uE4 * w / (dx*dx) */
  {
    size_t k = (size_t)src_z * nx + src_x;
    s->Ez[k] -= Cb[k] * w_n / (dx * dx);
  }
}

/* Magnetic update coefficient per cell: the paper's uH4 = 1/HA, HA = mu0 * mu_r / dt (ucget listing,
 * PAPER.md:291-295; model input `miu`, Table 1).  The listing indexes mr, uH1 and uH4 with
 * the same (i, j, k) as the H component they update, so the H component stored at array index (j, i) --
 * Hx at (j+1/2, i), Hy at (j, i+1/2) -- takes mu_r[j][i], without averaging (reading R22).
 * mu_r == NULL means mu_r = 1 everywhere (what every BASELINE.json config uses). */
static double *db_alloc(const oracle_params *p, const double *mu_r)
{
  const size_t ncell = (size_t)p->nz * p->nx;
  double *Db = (double *)malloc(ncell * sizeof(double));
  if (!Db) return NULL;
  for (size_t k = 0; k < ncell; ++k) Db[k] = p->dt / (MU0 * (mu_r ? mu_r[k] : 1.0));
  return Db;
}

static int check_geometry(const oracle_params *p, const int32_t *src_zx, const int32_t *rec_zx)
{
  if (p->nz < 3 || p->nx < 3 || p->nt <= 0 || p->nshots <= 0 || p->nrec < 0) return -1;
  if (p->nz < 2 * p->npml + 3 || p->nx < 2 * p->npml + 3) return -1;
  for (int s = 0; s < p->nshots; ++s) {
    int z = src_zx[2 * s], x = src_zx[2 * s + 1];
    if (z < 1 || z > p->nz - 2 || x < 1 || x > p->nx - 2) return -3;
    for (int r = 0; r < p->nrec; ++r) {
      z = rec_zx[((size_t)s * p->nrec + r) * 2];
      x = rec_zx[((size_t)s * p->nrec + r) * 2 + 1];
      if (z < 1 || z > p->nz - 2 || x < 1 || x > p->nx - 2) return -3;
    }
  }
  return 0;
}

/* ---------------------------------------------------------------------------------------
 * Forward modelling of all shots (Algorithm 1).
 *   traces   [nshots][nt][nrec]      traces[s][n][r] = Ez^n at receiver r (stage 1: recorded
 *                                    BEFORE step n, so sample 0 is 0; reading R8)
 *   ez_hist  NULL or [nshots][nt+1][nz][nx]      Ez^n, n = 0..nt  (stage 7)
 *   hx_hist  NULL or [nshots][nt+1][nz-1][nx]    Hx^{n-1/2}  (state at the start of step n)
 *   hy_hist  NULL or [nshots][nt+1][nz][nx-1]    Hy^{n-1/2}
 * returns 0, or <0 on bad arguments / out of memory.
 * ------------------------------------------------------------------------------------- */
int FN(forward)(const oracle_params *p, const SCALAR *eps_r, const SCALAR *sigma,
                const double *wavelet, const int32_t *src_zx, const int32_t *rec_zx,
                SCALAR *traces, SCALAR *ez_hist, SCALAR *hx_hist, SCALAR *hy_hist, const double *mu_r)
{
  int rc = check_geometry(p, src_zx, rec_zx);
  if (rc) return rc;
  const int nz = p->nz, nx = p->nx, nt = p->nt, R = p->nrec;
  const size_t ncell = (size_t)nz * nx;
  double *Db = db_alloc(p, mu_r);                /* uH4 */
  tables_t tab;
  if (!Db || tables_alloc(&tab, p)) { free(Db); return -4; }
  SCALAR *Ca = (SCALAR *)malloc(ncell * sizeof(SCALAR));
  SCALAR *Cb = (SCALAR *)malloc(ncell * sizeof(SCALAR));
  state_t st;
  SCALAR *buf = state_alloc(&st, nz, nx);
  if (!Ca || !Cb || !buf) { free(Ca); free(Cb); free(buf); free(Db); tables_free(&tab); return -4; }
  FN(coefficients)((int64_t)ncell, eps_r, sigma, p->dt, Ca, Cb);

  for (int s = 0; s < p->nshots; ++s) {
    memset(buf, 0, state_count(nz, nx) * sizeof(SCALAR));     /* fields zero at n = 0 */
    const double *w = wavelet + (p->wavelet_per_shot ? (size_t)s * nt : 0);
    const int32_t *rec = rec_zx + (size_t)s * R * 2;
    for (int n = 0; n < nt; ++n) {
      /* stage 1: save receivers data */
      for (int r = 0; r < R; ++r)
        traces[((size_t)s * nt + n) * R + r] = st.Ez[(size_t)rec[2 * r] * nx + rec[2 * r + 1]];
      /* stage 7 of the previous step == state at the start of this one */
      if (ez_hist) memcpy(ez_hist + ((size_t)s * (nt + 1) + n) * ncell, st.Ez, ncell * sizeof(SCALAR));
      if (hx_hist) memcpy(hx_hist + ((size_t)s * (nt + 1) + n) * (size_t)(nz - 1) * nx, st.Hx,
                          (size_t)(nz - 1) * nx * sizeof(SCALAR));
      if (hy_hist) memcpy(hy_hist + ((size_t)s * (nt + 1) + n) * (size_t)nz * (nx - 1), st.Hy,
                          (size_t)nz * (nx - 1) * sizeof(SCALAR));
      forward_step(&st, &tab, Ca, Cb, p->dx, Db, src_zx[2 * s], src_zx[2 * s + 1], w[n]);
    }
    if (ez_hist) memcpy(ez_hist + ((size_t)s * (nt + 1) + nt) * ncell, st.Ez, ncell * sizeof(SCALAR));
    if (hx_hist) memcpy(hx_hist + ((size_t)s * (nt + 1) + nt) * (size_t)(nz - 1) * nx, st.Hx,
                        (size_t)(nz - 1) * nx * sizeof(SCALAR));
    if (hy_hist) memcpy(hy_hist + ((size_t)s * (nt + 1) + nt) * (size_t)nz * (nx - 1), st.Hy,
                        (size_t)nz * (nx - 1) * sizeof(SCALAR));
  }
  free(Ca); free(Cb); free(buf); free(Db); tables_free(&tab);
  return 0;
}

#ifndef ORACLE_COMPLEX
/* ---------------------------------------------------------------------------------------
 * One reverse time step n of one shot: the transpose of forward_step, in Algorithm 2's
 * order: [gradient with the adjoint field of step n], transpose of the
 * electric update + electric PML, transpose of the magnetic update + magnetic PML, adjoint
 * source (residual sample n).  lam is the adjoint state (same layout as the forward state);
 * En = Ez^n, En1 = Ez^{n+1} from the forward history; gCa, gCb accumulate dJ/dCa, dJ/dCb.
 * Derivation: DESIGN.md section 4.
 * ------------------------------------------------------------------------------------- */
static void adjoint_step(state_t *lam, const tables_t *t, const double *Ca, const double *Cb,
                         double dx, const double *Db, const double *En, const double *En1,
                         double *gCa, double *gCb, double *tx, double *tz,
                         const int32_t *rec, int R, const double *res_n)
{
  const int nz = lam->nz, nx = lam->nx;
  /* 1. mask: the forward never updates the PEC ring, so nothing flows back through it */
  for (int i = 0; i < nx; ++i) { lam->Ez[i] = 0.0; lam->Ez[(size_t)(nz - 1) * nx + i] = 0.0; }
  for (int j = 0; j < nz; ++j) { lam->Ez[(size_t)j * nx] = 0.0; lam->Ez[(size_t)j * nx + nx - 1] = 0.0; }
  /* gradient w.r.t. the coefficients of step n (stage 6 of Algorithm 2; Eqs. 12-13 are the
   * dt -> 0 limit, reading R12).  E^{n+1} = Ca*E^n + Cb*(K - source) so the factor multiplying
   * Cb is (E^{n+1} - Ca*E^n)/Cb, which includes the source cell's term. */
#pragma omp parallel for schedule(static)
  for (int j = 1; j <= nz - 2; ++j)
    for (int i = 1; i <= nx - 2; ++i) {
      size_t k = (size_t)j * nx + i;
      gCa[k] += lam->Ez[k] * En[k];
      if (Cb[k] != 0.0) gCb[k] += lam->Ez[k] * (En1[k] - Ca[k] * En[k]) / Cb[k];
    }
  /* 2. transpose of the electric update + electric PML */
#pragma omp parallel for schedule(static)
  for (int j = 0; j < nz; ++j)
    for (int i = 0; i < nx; ++i) {
      size_t k = (size_t)j * nx + i;
      if (j == 0 || j == nz - 1 || i == 0 || i == nx - 1) { tx[k] = 0.0; tz[k] = 0.0; continue; }
      double q = Cb[k] * lam->Ez[k];
      double Tx = lam->pEzx[k] + q;
      tx[k] = q * t->ik_ex[i] + t->c_ex[i] * Tx;
      lam->pEzx[k] = t->b_ex[i] * Tx;
      double Tz = lam->pEzz[k] - q;
      tz[k] = -q * t->ik_ez[j] + t->c_ez[j] * Tz;
      lam->pEzz[k] = t->b_ez[j] * Tz;
      lam->Ez[k] = Ca[k] * lam->Ez[k];
    }
#pragma omp parallel for schedule(static)
  for (int j = 0; j < nz; ++j)
    for (int i = 0; i <= nx - 2; ++i)
      lam->Hy[(size_t)j * (nx - 1) + i] += (tx[(size_t)j * nx + i] - tx[(size_t)j * nx + i + 1]) / dx;
#pragma omp parallel for schedule(static)
  for (int j = 0; j <= nz - 2; ++j)
    for (int i = 0; i < nx; ++i)
      lam->Hx[(size_t)j * nx + i] += (tz[(size_t)j * nx + i] - tz[(size_t)(j + 1) * nx + i]) / dx;
  /* 3. transpose of the magnetic update + magnetic PML.  tx/tz are reused for sx/sz. */
#pragma omp parallel for schedule(static)
  for (int j = 0; j <= nz - 2; ++j)
    for (int i = 0; i < nx; ++i) {
      size_t k = (size_t)j * nx + i;
      double px = -Db[(size_t)j * nx + i] * lam->Hx[k];
      double T = lam->pHxz[k] + px;
      tz[k] = px * t->ik_hz[j] + t->c_hz[j] * T;        /* sz */
      lam->pHxz[k] = t->b_hz[j] * T;
    }
  for (int j = 0; j <= nz - 2; ++j)                      /* scatter: rows j and j+1 (serial) */
    for (int i = 0; i < nx; ++i) {
      double sz = tz[(size_t)j * nx + i];
      lam->Ez[(size_t)(j + 1) * nx + i] += sz / dx;
      lam->Ez[(size_t)j * nx + i] -= sz / dx;
    }
#pragma omp parallel for schedule(static)
  for (int j = 0; j < nz; ++j)
    for (int i = 0; i <= nx - 2; ++i) {
      size_t k = (size_t)j * (nx - 1) + i;
      double py = Db[(size_t)j * nx + i] * lam->Hy[k];
      double T = lam->pHyx[k] + py;
      double sx = py * t->ik_hx[i] + t->c_hx[i] * T;
      lam->pHyx[k] = t->b_hx[i] * T;
      tx[(size_t)j * nx + i] = sx;
    }
#pragma omp parallel for schedule(static)
  for (int j = 0; j < nz; ++j)
    for (int i = 0; i <= nx - 2; ++i) {                  /* scatter along the row (row-private) */
      double sx = tx[(size_t)j * nx + i];
      lam->Ez[(size_t)j * nx + i + 1] += sx / dx;
      lam->Ez[(size_t)j * nx + i] -= sx / dx;
    }
  /* 4. transpose of recording: adjoint source (stage 1 of Algorithm 2) */
  for (int r = 0; r < R; ++r)
    lam->Ez[(size_t)rec[2 * r] * nx + rec[2 * r + 1]] += res_n[r];
}

/* ---------------------------------------------------------------------------------------
 * Gradient of  sum_{s,n,r} residual*trace  (= J^T residual) w.r.t. eps_r and sigma on every
 * full-grid cell, summed over shots (Algorithm 2 + chain rule through Ca/Cb).
 *   residual [nshots][nt][nrec]
 *   checkpoint_stride = 0: the whole Ez history of a shot is kept ((nt+1) planes);
 *                     K > 0: the state is saved every K steps and each K-step segment is
 *                            recomputed before it is transposed (pin 9).
 *   traces may be NULL.
 * ------------------------------------------------------------------------------------- */
int oracle_gradient(const oracle_params *p, const double *eps_r, const double *sigma,
                    const double *wavelet, const int32_t *src_zx, const int32_t *rec_zx,
                    const double *residual, int checkpoint_stride,
                    double *traces, double *grad_eps_r, double *grad_sigma, const double *mu_r)
{
  int rc = check_geometry(p, src_zx, rec_zx);
  if (rc) return rc;
  const int nz = p->nz, nx = p->nx, nt = p->nt, R = p->nrec;
  const size_t ncell = (size_t)nz * nx;
  const size_t nstate = state_count(nz, nx);
  const int K = checkpoint_stride > 0 ? checkpoint_stride : nt;
  const int nseg = (nt + K - 1) / K;
  double *Db = db_alloc(p, mu_r);                /* uH4 per cell (mu_r == NULL: 1) */
  tables_t tab;
  if (!Db || tables_alloc(&tab, p)) { free(Db); return -4; }
  double *Ca = (double *)malloc(ncell * sizeof(double));
  double *Cb = (double *)malloc(ncell * sizeof(double));
  double *gCa = (double *)calloc(ncell, sizeof(double));
  double *gCb = (double *)calloc(ncell, sizeof(double));
  double *tx = (double *)malloc(ncell * sizeof(double));
  double *tz = (double *)malloc(ncell * sizeof(double));
  double *seg = (double *)malloc((size_t)(K + 1) * ncell * sizeof(double));  /* Ez^{cK..cK+K} */
  double *ckpt = (double *)malloc((size_t)nseg * nstate * sizeof(double));   /* state at n = cK */
  state_t st, lam;
  double *fbuf = state_alloc(&st, nz, nx);
  double *lbuf = state_alloc(&lam, nz, nx);
  if (!Ca || !Cb || !gCa || !gCb || !tx || !tz || !seg || !ckpt || !fbuf || !lbuf) {
    free(Ca); free(Cb); free(gCa); free(gCb); free(tx); free(tz); free(seg); free(ckpt);
    free(fbuf); free(lbuf); free(Db); tables_free(&tab);
    return -4;
  }
  oracle_coefficients((int64_t)ncell, eps_r, sigma, p->dt, Ca, Cb);

  for (int s = 0; s < p->nshots; ++s) {
    const double *w = wavelet + (p->wavelet_per_shot ? (size_t)s * nt : 0);
    const int32_t *rec = rec_zx + (size_t)s * R * 2;
    const double *res = residual + (size_t)s * nt * R;
    /* forward sweep, saving the state every K steps */
    memset(fbuf, 0, nstate * sizeof(double));
    for (int n = 0; n < nt; ++n) {
      if (traces)
        for (int r = 0; r < R; ++r)
          traces[((size_t)s * nt + n) * R + r] = st.Ez[(size_t)rec[2 * r] * nx + rec[2 * r + 1]];
      if (n % K == 0) memcpy(ckpt + (size_t)(n / K) * nstate, fbuf, nstate * sizeof(double));
      forward_step(&st, &tab, Ca, Cb, p->dx, Db, src_zx[2 * s], src_zx[2 * s + 1], w[n]);
    }
    /* reverse sweep, one segment at a time; lambda = 0 at the end time, Eq. (10) */
    memset(lbuf, 0, nstate * sizeof(double));
    for (int c = nseg - 1; c >= 0; --c) {
      int n0 = c * K, n1 = n0 + K < nt ? n0 + K : nt;
      memcpy(fbuf, ckpt + (size_t)c * nstate, nstate * sizeof(double));
      for (int n = n0; n < n1; ++n) {                      /* recompute Ez^{n0..n1} */
        memcpy(seg + (size_t)(n - n0) * ncell, st.Ez, ncell * sizeof(double));
        forward_step(&st, &tab, Ca, Cb, p->dx, Db, src_zx[2 * s], src_zx[2 * s + 1], w[n]);
      }
      memcpy(seg + (size_t)(n1 - n0) * ncell, st.Ez, ncell * sizeof(double));
      for (int n = n1 - 1; n >= n0; --n)
        adjoint_step(&lam, &tab, Ca, Cb, p->dx, Db, seg + (size_t)(n - n0) * ncell,
                     seg + (size_t)(n - n0 + 1) * ncell, gCa, gCb, tx, tz, rec, R, res + (size_t)n * R);
    }
  }
  /* chain rule Ca, Cb -> eps_r, sigma:
   *   dCa/d eps_r =  e0*sigma/dt / EA^2      dCb/d eps_r = -(e0/dt) / EA^2
   *   dCa/d sigma = -(e0*eps_r/dt) / EA^2    dCb/d sigma = -(1/2) / EA^2          */
  for (size_t k = 0; k < ncell; ++k) {
    if (sigma[k] > 100.0) { grad_eps_r[k] = 0.0; grad_sigma[k] = 0.0; continue; }
    double EA = EPS0 * eps_r[k] / p->dt + 0.5 * sigma[k];
    grad_eps_r[k] = EPS0 * (gCa[k] * (sigma[k] / p->dt) - gCb[k] * (1.0 / p->dt)) / (EA * EA);
    grad_sigma[k] = -(gCa[k] * (EPS0 * eps_r[k] / p->dt) + 0.5 * gCb[k]) / (EA * EA);
  }
  free(Ca); free(Cb); free(gCa); free(gCb); free(tx); free(tz); free(seg); free(ckpt);
  free(fbuf); free(lbuf); free(Db); tables_free(&tab);
  return 0;
}
#endif /* !ORACLE_COMPLEX */

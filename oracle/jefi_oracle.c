/*
 * jefi_oracle.c — TEST INFRASTRUCTURE, NOT PRODUCT.
 *
 * Plain, slow, fp64 CPU statement of what the JefiPIC hot path computes, written from
 * /root/reference/PAPER.md (arXiv 2209.07944) and the readings listed in DESIGN.md §3
 * (SURVEY.md §8(c) A1-A21).  It shares no code, header, table or constant with the CUDA
 * library under paper_2209_07944_b200/csrc; only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may load it.
 *
 * No blocking, fusion, tables or reordering: every (observation cell, source cell) pair is
 * evaluated in the order and notation of Eqs. (2.4)-(2.6); OpenMP only splits the independent
 * observation cells across threads.
 *
 * Layout conventions:
 *   cell index  c = i + nx*(j + ny*k)               (x fastest; reading A16)
 *   cell centre r = ((i+0.5)dx, (j+0.5)dy, (k+0.5)dz)   (Eq. 2.17 at :178)
 *   history     ring[slot][comp][c], comp = 0:rho 1:Jx 2:Jy 3:Jz, slot = step mod H,
 *               steps < 0 are zero, steps older than n-(H-1) are not stored and
 *               contribute zero (reading A15).
 *
 * Parity pins: tests/test_oracle_*.py (P1-P15 of SURVEY.md §8(c); P16 = the gamma of the Boris rotation when E and B are
 * both non-zero, hand-computed 90-degree rotations; L1-L6 for the linear retarded-time rule; Q1-Q7 in
 * tests/test_oracle_shape2.py for the S^(2) deposit / interpolation; F32 = orc_field_f32, the float-history instantiation of the
 * field body, bitwise against orc_field_f64 on the same values and against the dense enumeration,
 * tests/test_oracle_field.py::test_f32_history_entry_is_the_f64_entry_on_the_same_values); nothing here is "parity unpinned".
 */
#include <math.h>
#include <stddef.h>
#include <stdint.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORC_PI 3.14159265358979323846

int orc_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

void orc_set_num_threads(int n) {
#ifdef _OPENMP
  if (n > 0) omp_set_num_threads(n);
#else
  (void)n;
#endif
}

/* PAPER.md:211 (§2.4): N_dt = Ceiling(L_max/(c dt)), L_max the diagonal of the region (reading A17),
 * limited to hist_cap (N_dt = min(N_dt, 10000)). */
long orc_num_dt(int nx, int ny, int nz, double dx, double dy, double dz, double dt, double c, long hist_cap) {
  double lx = nx * dx, ly = ny * dy, lz = nz * dz;
  double lmax = sqrt(lx * lx + ly * ly + lz * lz);
  long ndt = (long)ceil(lmax / (c * dt));
  if (ndt > hist_cap) ndt = hist_cap;
  return ndt;
}

/* Eq. (2.6) with reading A1: the retarded time t^n - R/c is snapped to the NEAREST stored step,
 * m = floor(R/(c dt) + 1/2). */
long orc_delay(double ddx, double ddy, double ddz, double dt, double c) {
  double R = sqrt(ddx * ddx + ddy * ddy + ddz * ddz);
  double s = R / (c * dt);
  return (long)floor(s + 0.5);
}

/* Delay of every non-negative lattice offset (a, b, c) -> m_out[a + nx*(b + ny*c)].  Used by tests to
 * compare the device's delay table bit-exactly. */
void orc_delay_table(int nx, int ny, int nz, double dx, double dy, double dz, double dt, double c, int32_t* m_out) {
  for (int kc = 0; kc < nz; kc++)
    for (int jb = 0; jb < ny; jb++)
      for (int ia = 0; ia < nx; ia++)
        m_out[ia + (size_t)nx * (jb + (size_t)ny * kc)] = (int32_t)orc_delay(ia * dx, jb * dy, kc * dz, dt, c);
}

/* Retarded-time rules.  ORC_RULE_NEAREST is reading A1 (the five BASELINE.json configs): sources and derivatives taken
 * at the stored step nearest to t_r = t^n - R/c.  ORC_RULE_LINEAR is the second rule of SURVEY.md §8(f) NEXT-1 (reading
 * A22): the VALUES rho(t_r), J(t_r) of Eqs. (2.4)-(2.5) are taken on the straight line through the same
 * two samples that A1 uses, S(t_r) = S^{n-m} + (t_r - t^{n-m}) (S^{n-m} - S^{n-m-1})/dt with m the nearest step, i.e.
 * linear interpolation between steps n-m-1 and n-m when t_r falls between them and its continuation by up to dt/2
 * beyond step n-m otherwise (second-order accurate in dt); the time derivatives stay the paper's finite difference
 * (S^{n-m} - S^{n-m-1})/dt. */
#define ORC_RULE_NEAREST 0
#define ORC_RULE_LINEAR 1

/* ------------------------------------------------------------------------------------------------
 * Field: Eqs. (2.4)-(2.6); self cell skipped; zero before t0 (:217).
 * obs_idx == NULL -> all N cells (nobs must equal N).  E, B are [3][nobs] doubles.
 * The body is instantiated for a double and a float history (the float one only promotes on load).
 * ---------------------------------------------------------------------------------------------- */
#define ORC_FIELD_BODY(HT)                                                                                   \
  const size_t N = (size_t)nx * ny * nz;                                                                     \
  const double dV = dx * dy * dz;                                                                            \
  const double mu0 = 1.0 / (eps0 * c * c); /* reading A18 */                                                 \
  const double prefE = dV / (4.0 * ORC_PI * eps0);                                                           \
  const double prefB = -mu0 * dV / (4.0 * ORC_PI);                                                           \
  _Pragma("omp parallel for schedule(dynamic, 16)") for (long o = 0; o < nobs; o++) {                        \
    size_t oc = obs_idx ? (size_t)obs_idx[o] : (size_t)o;                                                    \
    int I = (int)(oc % nx), J = (int)((oc / nx) % ny), K = (int)(oc / ((size_t)nx * ny));                    \
    double Ex = 0, Ey = 0, Ez = 0, Bx = 0, By = 0, Bz = 0;                                                   \
    for (int k = 0; k < nz; k++)                                                                             \
      for (int j = 0; j < ny; j++)                                                                           \
        for (int i = 0; i < nx; i++) {                                                                       \
          if (i == I && j == J && k == K) continue;           /* PAPER.md:221 */                             \
          size_t sc = i + (size_t)nx * (j + (size_t)ny * k);                                                 \
          double ddx = (I - i) * dx, ddy = (J - j) * dy, ddz = (K - k) * dz; /* r - r' */                    \
          double R2 = ddx * ddx + ddy * ddy + ddz * ddz;                                                     \
          double R = sqrt(R2);                                                                               \
          double s = R / (c * dt);                               /* Eq. (2.6) */                             \
          long m = (long)floor(s + 0.5);                         /* reading A1 */                            \
          if (m > (long)H - 2) continue;                         /* reading A15 */                           \
          long t0 = (long)n - m, t1 = t0 - 1;                                                                \
          double rho0 = 0, jx0 = 0, jy0 = 0, jz0 = 0, rho1 = 0, jx1 = 0, jy1 = 0, jz1 = 0;                   \
          if (t0 >= 0) {                                         /* PAPER.md:217 */                          \
            const HT* S = ring + (size_t)(t0 % H) * 4 * N;                                                   \
            rho0 = S[sc]; jx0 = S[N + sc]; jy0 = S[2 * N + sc]; jz0 = S[3 * N + sc];                         \
          }                                                                                                  \
          if (t1 >= 0) {                                                                                     \
            const HT* S = ring + (size_t)(t1 % H) * 4 * N;                                                   \
            rho1 = S[sc]; jx1 = S[N + sc]; jy1 = S[2 * N + sc]; jz1 = S[3 * N + sc];                         \
          }                                                                                                  \
          double drho = (rho0 - rho1) / dt;                      /* backward difference, Eq. (2.4) */        \
          double djx = (jx0 - jx1) / dt, djy = (jy0 - jy1) / dt, djz = (jz0 - jz1) / dt; /* Eq. (2.5) */     \
          if (rule == ORC_RULE_LINEAR) { /* reading A22: S(t_r) = S^{n-m} + (t_r - t^{n-m}) S_dot^{n-m} */   \
            double tr_minus_tm = ((double)m - s) * dt;           /* t_r = t^n - s dt, t^{n-m} = t^n - m dt */   \
            rho0 += tr_minus_tm * drho;                                                                      \
            jx0 += tr_minus_tm * djx; jy0 += tr_minus_tm * djy; jz0 += tr_minus_tm * djz;                    \
          }                                                                                                  \
          double R3 = R2 * R;                                                                                \
          /* Eq. (2.4): d rho/R^3 + d rho_dot/(c R^2) - J_dot/(c^2 R)   (reading A2) */                      \
          Ex += ddx * rho0 / R3 + ddx * drho / (c * R2) - djx / (c * c * R);                                 \
          Ey += ddy * rho0 / R3 + ddy * drho / (c * R2) - djy / (c * c * R);                                 \
          Ez += ddz * rho0 / R3 + ddz * drho / (c * R2) - djz / (c * c * R);                                 \
          /* Eq. (2.5): d x ( J/R^3 + J_dot/(c R^2) )   (reading A3) */                                      \
          double wx = jx0 / R3 + djx / (c * R2);                                                             \
          double wy = jy0 / R3 + djy / (c * R2);                                                             \
          double wz = jz0 / R3 + djz / (c * R2);                                                             \
          Bx += ddy * wz - ddz * wy;                                                                         \
          By += ddz * wx - ddx * wz;                                                                         \
          Bz += ddx * wy - ddy * wx;                                                                         \
        }                                                                                                    \
    E[o] = prefE * Ex; E[nobs + o] = prefE * Ey; E[2 * nobs + o] = prefE * Ez;                               \
    B[o] = prefB * Bx; B[nobs + o] = prefB * By; B[2 * nobs + o] = prefB * Bz;                               \
  }

void orc_field_f64(int nx, int ny, int nz, double dx, double dy, double dz, double dt, double c, double eps0, int rule,
                   long n, long H, const double* ring, long nobs, const int64_t* obs_idx, double* E, double* B) {
  ORC_FIELD_BODY(double)
}

void orc_field_f32(int nx, int ny, int nz, double dx, double dy, double dz, double dt, double c, double eps0, int rule,
                   long n, long H, const float* ring, long nobs, const int64_t* obs_idx, double* E, double* B) {
  ORC_FIELD_BODY(float)
}

/* ------------------------------------------------------------------------------------------------
 * Cell index and fractions, Eqs. (2.15), (2.17) (reading A9: floor).
 * Positions are in grid units xi = x/dx, so i = floor(xi - 0.5), alpha = xi - 0.5 - i.
 * ---------------------------------------------------------------------------------------------- */
static inline void orc_cell(double xi, long* i, double* alpha) {
  double s = xi - 0.5;
  double f = floor(s);
  *i = (long)f;
  *alpha = s - f;
}

void orc_cell_index(long np, const double* x, const double* y, const double* z, int32_t* ijk /* [np][3] */) {
  for (long p = 0; p < np; p++) {
    long i, j, k; double a;
    orc_cell(x[p], &i, &a); orc_cell(y[p], &j, &a); orc_cell(z[p], &k, &a);
    ijk[3 * p] = (int32_t)i; ijk[3 * p + 1] = (int32_t)j; ijk[3 * p + 2] = (int32_t)k;
  }
}

/* CIC deposit, Eqs. (2.15)-(2.19), all 8 weights (reading A10); nodes outside the
 * region are virtual and are not stored (reading A8).  u = gamma v / c, so
 * v = c u / sqrt(1+|u|^2).  Dead particles are not sources (reading A13).
 * rho, jx, jy, jz: N doubles each, overwritten.  Serial, particle order, plain sums. */
void orc_deposit(int nx, int ny, int nz, double dx, double dy, double dz, double c, long np,
                 const double* x, const double* y, const double* z,
                 const double* ux, const double* uy, const double* uz,
                 const double* qw, const uint8_t* alive,
                 double* rho, double* jx, double* jy, double* jz) {
  const size_t N = (size_t)nx * ny * nz;
  const double dV = dx * dy * dz;
  for (size_t cidx = 0; cidx < N; cidx++) { rho[cidx] = 0; jx[cidx] = 0; jy[cidx] = 0; jz[cidx] = 0; }
  for (long p = 0; p < np; p++) {
    if (alive && !alive[p]) continue;
    long i, j, k; double al, be, ch;
    orc_cell(x[p], &i, &al); orc_cell(y[p], &j, &be); orc_cell(z[p], &k, &ch);   /* Eqs. (2.15), (2.17) */
    double g = sqrt(1.0 + ux[p] * ux[p] + uy[p] * uy[p] + uz[p] * uz[p]);
    double vx = c * ux[p] / g, vy = c * uy[p] / g, vz = c * uz[p] / g;
    for (int cc = 0; cc < 2; cc++)
      for (int bb = 0; bb < 2; bb++)
        for (int aa = 0; aa < 2; aa++) {
          long ii = i + aa, jj = j + bb, kk = k + cc;
          if (ii < 0 || ii >= nx || jj < 0 || jj >= ny || kk < 0 || kk >= nz) continue; /* virtual node */
          double w = (aa ? al : 1.0 - al) * (bb ? be : 1.0 - be) * (cc ? ch : 1.0 - ch); /* Eq. (2.16) */
          double r = qw[p] * w / dV;                                                    /* Eq. (2.18) */
          size_t cidx = ii + (size_t)nx * (jj + (size_t)ny * kk);
          rho[cidx] += r;
          jx[cidx] += r * vx; jy[cidx] += r * vy; jz[cidx] += r * vz;                    /* Eq. (2.19) */
        }
  }
}

/* Field interpolation to one particle, Eq. (2.20): same 8 weights; fields at virtual
 * nodes are zero and the weights are not renormalised (reading A12). */
static void orc_gather(int nx, int ny, int nz, double xi, double eta, double zeta,
                       const double* fx, const double* fy, const double* fz, double out[3]) {
  long i, j, k; double al, be, ch;
  orc_cell(xi, &i, &al); orc_cell(eta, &j, &be); orc_cell(zeta, &k, &ch);
  out[0] = out[1] = out[2] = 0;
  for (int cc = 0; cc < 2; cc++)
    for (int bb = 0; bb < 2; bb++)
      for (int aa = 0; aa < 2; aa++) {
        long ii = i + aa, jj = j + bb, kk = k + cc;
        if (ii < 0 || ii >= nx || jj < 0 || jj >= ny || kk < 0 || kk >= nz) continue;
        double w = (aa ? al : 1.0 - al) * (bb ? be : 1.0 - be) * (cc ? ch : 1.0 - ch);
        size_t cidx = ii + (size_t)nx * (jj + (size_t)ny * kk);
        out[0] += w * fx[cidx]; out[1] += w * fy[cidx]; out[2] += w * fz[cidx];
      }
}

/* ------------------------------------------------------------------------------------------------
 * Second-order shape function S^(2), Eq. (2.14) with reading A11: the printed
 * first range "0 <= |x| <= Delta" overlaps the second and must read 0 <= |x| <= Delta/2 (the two branches then meet at
 * |x| = Delta/2 with value 1/2 and S^(2) is the quadratic B-spline):
 *     S2(x) = (1/Delta^2) (-x^2 + 3/4 Delta^2)          for        |x| <= Delta/2
 *           = (1/(8 Delta^2)) (2|x| - 3 Delta)^2        for Delta/2 <= |x| <= 3/2 Delta,      0 beyond.
 * the same allocation as Eqs. (2.16)-(2.20) with S^(2) in place of the linear weights.
 * A particle at xi (grid units, Delta = 1) lies in cell ic = floor(xi) whose centre is at ic + 1/2; the centres within
 * 3/2 of it are ic-1, ic, ic+1, so 3 nodes per axis (27 in 3-D) get weight S2(xi - (node + 1/2)); the weight of node
 * (a, b, c) is the product of the three axis weights, as for the volume weighting of Eq. (2.16).  Nodes outside the region
 * are virtual and dropped / count as zero exactly as for first order (readings A8, A12).
 * ---------------------------------------------------------------------------------------------- */
static double orc_s2(double x) {
  double ax = fabs(x);
  if (ax <= 0.5) return -x * x + 0.75;
  if (ax <= 1.5) return (2.0 * ax - 3.0) * (2.0 * ax - 3.0) / 8.0;
  return 0.0;
}

/* the three nodes ic-1, ic, ic+1 of one axis and their weights */
static inline void orc_cell_s2(double xi, long* ic, double w[3]) {
  double f = floor(xi);
  *ic = (long)f;
  for (int a = -1; a <= 1; a++) w[a + 1] = orc_s2(xi - ((double)(*ic + a) + 0.5));
}

void orc_cell_index_s2(long np, const double* x, const double* y, const double* z, int32_t* ijk /* [np][3], centre node */) {
  for (long p = 0; p < np; p++) {
    ijk[3 * p] = (int32_t)floor(x[p]); ijk[3 * p + 1] = (int32_t)floor(y[p]); ijk[3 * p + 2] = (int32_t)floor(z[p]);
  }
}

void orc_deposit_s2(int nx, int ny, int nz, double dx, double dy, double dz, double c, long np,
                    const double* x, const double* y, const double* z,
                    const double* ux, const double* uy, const double* uz,
                    const double* qw, const uint8_t* alive,
                    double* rho, double* jx, double* jy, double* jz) {
  const size_t N = (size_t)nx * ny * nz;
  const double dV = dx * dy * dz;
  for (size_t cidx = 0; cidx < N; cidx++) { rho[cidx] = 0; jx[cidx] = 0; jy[cidx] = 0; jz[cidx] = 0; }
  for (long p = 0; p < np; p++) {
    if (alive && !alive[p]) continue;
    long i, j, k; double wx[3], wy[3], wz[3];
    orc_cell_s2(x[p], &i, wx); orc_cell_s2(y[p], &j, wy); orc_cell_s2(z[p], &k, wz);
    double g = sqrt(1.0 + ux[p] * ux[p] + uy[p] * uy[p] + uz[p] * uz[p]);
    double vx = c * ux[p] / g, vy = c * uy[p] / g, vz = c * uz[p] / g;
    for (int cc = -1; cc <= 1; cc++)
      for (int bb = -1; bb <= 1; bb++)
        for (int aa = -1; aa <= 1; aa++) {
          long ii = i + aa, jj = j + bb, kk = k + cc;
          if (ii < 0 || ii >= nx || jj < 0 || jj >= ny || kk < 0 || kk >= nz) continue; /* virtual node */
          double w = wx[aa + 1] * wy[bb + 1] * wz[cc + 1];
          double r = qw[p] * w / dV;                                                    /* Eq. (2.18) */
          size_t cidx = ii + (size_t)nx * (jj + (size_t)ny * kk);
          rho[cidx] += r;
          jx[cidx] += r * vx; jy[cidx] += r * vy; jz[cidx] += r * vz;                    /* Eq. (2.19) */
        }
  }
}

static void orc_gather_s2(int nx, int ny, int nz, double xi, double eta, double zeta,
                          const double* fx, const double* fy, const double* fz, double out[3]) {
  long i, j, k; double wx[3], wy[3], wz[3];
  orc_cell_s2(xi, &i, wx); orc_cell_s2(eta, &j, wy); orc_cell_s2(zeta, &k, wz);
  out[0] = out[1] = out[2] = 0;
  for (int cc = -1; cc <= 1; cc++)
    for (int bb = -1; bb <= 1; bb++)
      for (int aa = -1; aa <= 1; aa++) {
        long ii = i + aa, jj = j + bb, kk = k + cc;
        if (ii < 0 || ii >= nx || jj < 0 || jj >= ny || kk < 0 || kk >= nz) continue;
        double w = wx[aa + 1] * wy[bb + 1] * wz[cc + 1];
        size_t cidx = ii + (size_t)nx * (jj + (size_t)ny * kk);
        out[0] += w * fx[cidx]; out[1] += w * fy[cidx]; out[2] += w * fz[cidx];
      }
}

void orc_interp_s2(int nx, int ny, int nz, long np, const double* x, const double* y, const double* z,
                   const double* fx, const double* fy, const double* fz, double* out /* [np][3] */) {
  for (long p = 0; p < np; p++) orc_gather_s2(nx, ny, nz, x[p], y[p], z[p], fx, fy, fz, out + 3 * p);
}

void orc_interp(int nx, int ny, int nz, long np, const double* x, const double* y, const double* z,
                const double* fx, const double* fy, const double* fz, double* out /* [np][3] */) {
  for (long p = 0; p < np; p++) orc_gather(nx, ny, nz, x[p], y[p], z[p], fx, fy, fz, out + 3 * p);
}

/* Interpolation + Boris push + kill.  Eqs. (2.7)-(2.11) in the relativistic form of
 * readings A5/A6 (u = gamma v/c; identical to the paper's printed form as gamma -> 1), position update
 * Eq. (2.8), kill rule PAPER.md:205, 239 (reading A13).  Given momenta are u^{n-1/2} (reading A7).
 * Eext/Bext are uniform background fields added at the particle.
 * Positions in grid units, updated in place; alive[p] cleared when the particle leaves [0,n) on any axis.
 * shape_order: 1 = the paper's linear weights (Eq. 2.20), 2 = S^(2) (Eq. 2.14). */
void orc_push(int nx, int ny, int nz, double dx, double dy, double dz, double dt, double c, long np,
              double* x, double* y, double* z, double* ux, double* uy, double* uz,
              const double* q_over_m, uint8_t* alive,
              const double* ex, const double* ey, const double* ez,
              const double* bx, const double* by, const double* bz,
              const double* Eext, const double* Bext, int shape_order) {
  for (long p = 0; p < np; p++) {
    if (!alive[p]) continue;
    double Ep[3], Bp[3];
    if (shape_order == 2) {                                        /* S^(2) weights, Eq. (2.14) */
      orc_gather_s2(nx, ny, nz, x[p], y[p], z[p], ex, ey, ez, Ep);
      orc_gather_s2(nx, ny, nz, x[p], y[p], z[p], bx, by, bz, Bp);
    } else {
      orc_gather(nx, ny, nz, x[p], y[p], z[p], ex, ey, ez, Ep);   /* Eq. (2.20) */
      orc_gather(nx, ny, nz, x[p], y[p], z[p], bx, by, bz, Bp);
    }
    for (int a = 0; a < 3; a++) { Ep[a] += Eext[a]; Bp[a] += Bext[a]; }
    double h = q_over_m[p] * dt / 2.0;
    /* Eq. (2.9): half electric kick */
    double umx = ux[p] + h * Ep[0] / c, umy = uy[p] + h * Ep[1] / c, umz = uz[p] + h * Ep[2] / c;
    /* Eq. (2.10): rotation about B with gamma of u^- */
    double gm = sqrt(1.0 + umx * umx + umy * umy + umz * umz);
    double tx = h * Bp[0] / gm, ty = h * Bp[1] / gm, tz = h * Bp[2] / gm;
    double upx = umx + (umy * tz - umz * ty);
    double upy = umy + (umz * tx - umx * tz);
    double upz = umz + (umx * ty - umy * tx);
    double t2 = tx * tx + ty * ty + tz * tz;
    double sx = 2.0 * tx / (1.0 + t2), sy = 2.0 * ty / (1.0 + t2), sz = 2.0 * tz / (1.0 + t2);
    double uqx = umx + (upy * sz - upz * sy);
    double uqy = umy + (upz * sx - upx * sz);
    double uqz = umz + (upx * sy - upy * sx);
    /* Eq. (2.11): second half electric kick */
    double unx = uqx + h * Ep[0] / c, uny = uqy + h * Ep[1] / c, unz = uqz + h * Ep[2] / c;
    double gn = sqrt(1.0 + unx * unx + uny * uny + unz * unz);
    double vx = c * unx / gn, vy = c * uny / gn, vz = c * unz / gn;
    /* Eq. (2.8) in grid units */
    double xn = x[p] + vx * dt / dx, yn = y[p] + vy * dt / dy, zn = z[p] + vz * dt / dz;
    ux[p] = unx; uy[p] = uny; uz[p] = unz;
    x[p] = xn; y[p] = yn; z[p] = zn;
    if (xn < 0.0 || xn >= (double)nx || yn < 0.0 || yn >= (double)ny || zn < 0.0 || zn >= (double)nz) alive[p] = 0;
  }
}

// cuth_oracle.cpp -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
//
// Plain, slow, fp64 CPU oracle for the hot path of CUTh-Solver (arxiv/paper_2606_17850):
// Jacobi-preconditioned Conjugate Gradient on the SPD 7-point finite-volume thermal system.
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
// call this.  It shares no source, header, table or helper with paper_2606_17850_b200/csrc.
//
// What each function follows (PAPER.md = /root/reference/PAPER.md at survey time):
//   oracle_assemble_csr   eq. (4) steady balance and eq. (5) backward Euler
//                         (PAPER.md:130-133), cell by cell, into CSR (the paper's "CSR baseline",
//                         PAPER.md:495).  Adiabatic faces emit nothing (eq. (3));
//                         the Robin top adds h*S to the diagonal (eq. (2)/(4)).
//                         Face conductance = series of two half cells (harmonic mean; R1).
//   oracle_csr_spmv       y = A x, the definition (row loop, left-to-right in stored column order).
//   oracle_csr_to_dia     Quad-Diag layout of PAPER.md:219 and Alg. 2's slice lengths
//                         (PAPER.md:192-215): 4 unpadded upper diagonals, read off the CSR.
//   oracle_pcg            Alg. 1 step by step, M = diag(A) (Jacobi, PAPER.md:231,
//                         586) or M = I; stopping rule relative, verified on b - A x (R7).
//   oracle_cheb_apply / oracle_lanczos / oracle_pcg_cheb   Alg. 3, Lanczos
//                         and Alg. 1 with M^-1 = Alg. 3: the paper's own preconditioner.
//   oracle_transient_rhs  right-hand side of eq. (5): b = P_{n+1} + (C V / dt) T_n  (T_amb = 0).
//
// Pins (tests/test_oracle_*.py, -m "not gpu"): closed-form 1-D slab profile, dense Cholesky on
// tiny grids, separable direct solve (DCT + Thomas), A*1 = s row sums, symmetry / sign
// invariants, nnz and layout closed forms, energy balance, CG monotonicity of the A-norm error.
//
// Build: g++ -O2 -fopenmp -ffp-contract=off -shared -fPIC (oracle/build.py).  No FMA contraction so
// that the matrix entries are the plainly rounded result of the written expressions.

#include <cmath>
#include <cstdint>
#include <cstring>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

inline int64_t lin(int64_t x, int64_t y, int64_t z, int64_t nx, int64_t ny) { return x + nx * (y + ny * z); }

struct Grid {
  int64_t nx, ny, nz;
  double dx, dy;
  const double* dz;
  const double* kappa;
  int per_layer;
  double kap(int64_t x, int64_t y, int64_t z) const { return per_layer ? kappa[z] : kappa[lin(x, y, z, nx, ny)]; }
  // series of two half-cell resistances between neighbouring cell centres, a = lower-index cell
  double gx(int64_t x, int64_t y, int64_t z) const {  // between (x,y,z) and (x+1,y,z)
    double ka = kap(x, y, z), kb = kap(x + 1, y, z);
    return (dy * dz[z]) / (dx / (2.0 * ka) + dx / (2.0 * kb));
  }
  double gy(int64_t x, int64_t y, int64_t z) const {  // between (x,y,z) and (x,y+1,z)
    double ka = kap(x, y, z), kb = kap(x, y + 1, z);
    return (dx * dz[z]) / (dy / (2.0 * ka) + dy / (2.0 * kb));
  }
  double gz(int64_t x, int64_t y, int64_t z) const {  // between (x,y,z) and (x,y,z+1)
    double ka = kap(x, y, z), kb = kap(x, y, z + 1);
    return (dx * dy) / (dz[z] / (2.0 * ka) + dz[z + 1] / (2.0 * kb));
  }
};

double dot(int64_t n, const double* a, const double* b) {
  double s = 0.0;
#pragma omp parallel for reduction(+ : s) schedule(static)
  for (int64_t i = 0; i < n; ++i) s += a[i] * b[i];
  return s;
}

void spmv(int64_t n, const int64_t* rp, const int32_t* ci, const double* v, const double* x, double* y) {
#pragma omp parallel for schedule(static)
  for (int64_t i = 0; i < n; ++i) {
    double s = 0.0;
    for (int64_t k = rp[i]; k < rp[i + 1]; ++k) s += v[k] * x[ci[k]];
    y[i] = s;
  }
}

}  // namespace

extern "C" {

int oracle_num_threads() {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

// nnz of the 7-point matrix with adiabatic sides: 7N - 2(nx ny + nx nz + ny nz)
int64_t oracle_csr_nnz(int64_t nx, int64_t ny, int64_t nz) {
  return 7 * nx * ny * nz - 2 * (nx * ny + nx * nz + ny * nz);
}

// eq. (4)/(5).  rowptr[N+1], col[nnz] ascending within a row, val[nnz].
// cvol == nullptr or dt <= 0  =>  steady.  kappa: nz values (per_layer != 0) or N values.
int oracle_assemble_csr(int64_t nx, int64_t ny, int64_t nz, double dx, double dy, const double* dz,
                        const double* kappa, int kappa_is_per_layer, double h_top, const double* cvol,
                        double dt, int64_t* rowptr, int32_t* col, double* val) {
  if (nx < 1 || ny < 1 || nz < 1) return -1;
  Grid g{nx, ny, nz, dx, dy, dz, kappa, kappa_is_per_layer};
  const int64_t n = nx * ny * nz;
  const bool transient = (cvol != nullptr) && dt > 0.0;
  // pass 1: row lengths
  rowptr[0] = 0;
  for (int64_t z = 0; z < nz; ++z)
    for (int64_t y = 0; y < ny; ++y)
      for (int64_t x = 0; x < nx; ++x) {
        int c = 1 + (z > 0) + (y > 0) + (x > 0) + (x + 1 < nx) + (y + 1 < ny) + (z + 1 < nz);
        int64_t i = lin(x, y, z, nx, ny);
        rowptr[i + 1] = rowptr[i] + c;
      }
#pragma omp parallel for schedule(static) collapse(2)
  for (int64_t z = 0; z < nz; ++z)
    for (int64_t y = 0; y < ny; ++y)
      for (int64_t x = 0; x < nx; ++x) {
        const int64_t i = lin(x, y, z, nx, ny);
        int64_t k = rowptr[i];
        double diag = 0.0;
        int64_t kd = -1;
        // ascending column order: -z, -y, -x, diag, +x, +y, +z
        if (z > 0) { double c = g.gz(x, y, z - 1); col[k] = (int32_t)lin(x, y, z - 1, nx, ny); val[k++] = -c; diag = diag + c; }
        if (y > 0) { double c = g.gy(x, y - 1, z); col[k] = (int32_t)lin(x, y - 1, z, nx, ny); val[k++] = -c; diag = diag + c; }
        if (x > 0) { double c = g.gx(x - 1, y, z); col[k] = (int32_t)lin(x - 1, y, z, nx, ny); val[k++] = -c; diag = diag + c; }
        kd = k; col[k++] = (int32_t)i;
        if (x + 1 < nx) { double c = g.gx(x, y, z); col[k] = (int32_t)lin(x + 1, y, z, nx, ny); val[k++] = -c; diag = diag + c; }
        if (y + 1 < ny) { double c = g.gy(x, y, z); col[k] = (int32_t)lin(x, y + 1, z, nx, ny); val[k++] = -c; diag = diag + c; }
        if (z + 1 < nz) { double c = g.gz(x, y, z); col[k] = (int32_t)lin(x, y, z + 1, nx, ny); val[k++] = -c; diag = diag + c; }
        if (z == nz - 1) diag = diag + h_top * (dx * dy);                      // Robin top, hS_0 T_0
        if (transient) diag = diag + cvol[z] * ((dx * dy) * dz[z]) / dt;       // C_0 V_0 / dt
        val[kd] = diag;
      }
  (void)n;
  return 0;
}

void oracle_csr_spmv(int64_t n, const int64_t* rowptr, const int32_t* col, const double* val, const double* x,
                     double* y) {
  spmv(n, rowptr, col, val, x, y);
}

// Condensed DIA ("Quad-Diag"): diagonal k (offsets 0, 1, nx, nx*ny) has exactly
// N - o_k elements, element j = A[j, j + o_k]; absent entries are +0.0.  Packed D0|D1|D2|D3.
int oracle_csr_to_dia(int64_t nx, int64_t ny, int64_t nz, const int64_t* rowptr, const int32_t* col,
                      const double* val, double* vals, int64_t* ptr5, int64_t* off4) {
  const int64_t n = nx * ny * nz;
  off4[0] = 0; off4[1] = 1; off4[2] = nx; off4[3] = nx * ny;
  ptr5[0] = 0;
  for (int k = 0; k < 4; ++k) ptr5[k + 1] = ptr5[k] + (n - off4[k]);
  for (int k = 0; k < 4; ++k) {
    const int64_t o = off4[k];
    for (int64_t j = 0; j + o < n; ++j) {
      double v = 0.0;
      for (int64_t q = rowptr[j]; q < rowptr[j + 1]; ++q)
        if ((int64_t)col[q] == j + o) v = val[q];
      vals[ptr5[k] + j] = v;
    }
  }
  return 0;
}

// rhs of eq. (5) with T_amb = 0:  b_i = P_i + (C_z V_z / dt) T_i
void oracle_transient_rhs(int64_t nx, int64_t ny, int64_t nz, double dx, double dy, const double* dz,
                          const double* cvol, double dt, const double* power, const double* t_n, double* b) {
  for (int64_t z = 0; z < nz; ++z) {
    const double cap = cvol[z] * ((dx * dy) * dz[z]) / dt;
    for (int64_t q = 0; q < nx * ny; ++q) {
      const int64_t i = z * nx * ny + q;
      b[i] = power[i] + cap * t_n[i];
    }
  }
}

// Alg. 1.  precond: 0 => M = I, 1 => M = diag(A).
// x: in x_0, out x_k.  Stop when ||r||_2 <= rtol ||b||_2 on the recursive r AND on a fresh b - A x
// (if the fresh one fails: r = fresh, z = M^-1 r, p = z, continue).  b = 0 => x = 0.
// hist (nullable, length hist_len): hist[k] = ||r_k||_2 / ||b||_2 of the recursive residual.
// Returns 0 converged, 1 max_iters reached, 2 breakdown (p'Ap <= 0 or non-finite).
int oracle_pcg(int64_t n, const int64_t* rowptr, const int32_t* col, const double* val, const double* b,
               double* x, double rtol, int64_t max_iters, int precond, int64_t* iters_out,
               double* relres_true_out, double* hist, int64_t hist_len) {
  std::vector<double> r(n), z(n), p(n), mu(n), dg(n);
  for (int64_t i = 0; i < n; ++i) {
    double d = 1.0;
    if (precond == 1)
      for (int64_t k = rowptr[i]; k < rowptr[i + 1]; ++k)
        if ((int64_t)col[k] == i) d = val[k];
    dg[i] = d;
  }
  const double bnorm = std::sqrt(dot(n, b, b));
  int64_t it = 0;
  int status = 1;
  if (bnorm == 0.0) {
    std::memset(x, 0, sizeof(double) * n);
    *iters_out = 0;
    *relres_true_out = 0.0;
    return 0;
  }
  const double tol = rtol * bnorm;
  spmv(n, rowptr, col, val, x, mu.data());                                  // line 1: r0 = b - A x0
  for (int64_t i = 0; i < n; ++i) r[i] = b[i] - mu[i];
  for (int64_t i = 0; i < n; ++i) z[i] = r[i] / dg[i];                      // line 2
  p = z;                                                                    // line 3
  double rho = dot(n, r.data(), z.data());
  double rnorm = std::sqrt(dot(n, r.data(), r.data()));
  if (hist && 0 < hist_len) hist[0] = rnorm / bnorm;
  double rel_true = rnorm / bnorm;
  for (;;) {
    if (rnorm <= tol) {                                                     // line 5 + verification
      spmv(n, rowptr, col, val, x, mu.data());
      for (int64_t i = 0; i < n; ++i) mu[i] = b[i] - mu[i];
      const double tn = std::sqrt(dot(n, mu.data(), mu.data()));
      rel_true = tn / bnorm;
      if (tn <= tol) { status = 0; break; }
      r = mu;
      for (int64_t i = 0; i < n; ++i) z[i] = r[i] / dg[i];
      p = z;
      rho = dot(n, r.data(), z.data());
      rnorm = tn;
    }
    if (it >= max_iters) { status = 1; break; }
    spmv(n, rowptr, col, val, p.data(), mu.data());                         // line 6
    const double pmu = dot(n, p.data(), mu.data());
    if (!(pmu > 0.0) || !std::isfinite(pmu) || !std::isfinite(rho)) { status = 2; break; }
    const double alpha = rho / pmu;                                         // line 7
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n; ++i) {
      x[i] += alpha * p[i];                                                 // line 8
      r[i] -= alpha * mu[i];                                                // line 9
      z[i] = r[i] / dg[i];                                                  // line 10
    }
    const double rho_new = dot(n, r.data(), z.data());
    const double beta = rho_new / rho;                                      // line 11
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n; ++i) p[i] = z[i] + beta * p[i];              // line 12
    rho = rho_new;
    rnorm = std::sqrt(dot(n, r.data(), r.data()));
    ++it;                                                                   // line 13
    if (hist && it < hist_len) hist[it] = rnorm / bnorm;
  }
  if (status != 0) {
    spmv(n, rowptr, col, val, x, mu.data());
    for (int64_t i = 0; i < n; ++i) mu[i] = b[i] - mu[i];
    rel_true = std::sqrt(dot(n, mu.data(), mu.data())) / bnorm;
  }
  *iters_out = it;
  *relres_true_out = rel_true;
  return status;
}

// Run exactly `iters` iterations of Alg. 1 lines 6-13 from x (no convergence test): used only to
// time a fixed window of the oracle on grids where a full solve takes hours (bench.py cpu_baseline).
void oracle_pcg_window(int64_t n, const int64_t* rowptr, const int32_t* col, const double* val, const double* b,
                       double* x, int64_t iters, int precond) {
  int64_t it;
  double rel;
  oracle_pcg(n, rowptr, col, val, b, x, 0.0, iters, precond, &it, &rel, nullptr, 0);
}

// ---------------------------------------------------------------------------------------------
// NEXT-1: the paper's own preconditioner.
//
// Alg. 3, Chebyshev polynomial preconditioning, step by step in the paper's order,
// with the readings of DESIGN.md R-G16 for its garbles: z starts at 0, line 9 reads 2*sigma_1, and
// rho_0 = 1/sigma_1 = delta/theta (PAPER.md:286 and 311 agree).  theta, delta from eq. (11b).
// z = q(A) r with 1 - lambda q(lambda) = C_k((theta-lambda)/delta) / C_k(theta/delta)  (eq. (11a)).
void oracle_cheb_apply(int64_t n, const int64_t* rowptr, const int32_t* col, const double* val, const double* r,
                       double lmin, double lmax, int k, double* z) {
  std::vector<double> rc(r, r + n), d(n), ad(n);
  const double theta = (lmax + lmin) / 2.0, delta = (lmax - lmin) / 2.0;       // eq. (11b)
  const double sigma1 = theta / delta;                                         // line 2
  double rho = 1.0 / sigma1;                                                   // line 3
  for (int64_t i = 0; i < n; ++i) { d[i] = rc[i] / theta; z[i] = 0.0; }        // line 4 (z = 0: R-G16)
  for (int it = 0; it < k; ++it) {                                             // line 5
    for (int64_t i = 0; i < n; ++i) z[i] = z[i] + d[i];                        // line 6
    spmv(n, rowptr, col, val, d.data(), ad.data());                            // line 7
    for (int64_t i = 0; i < n; ++i) rc[i] = rc[i] - ad[i];                     // line 8
    const double rho_next = 1.0 / (2.0 * sigma1 - rho);                        // line 9
    for (int64_t i = 0; i < n; ++i) d[i] = rho_next * rho * d[i] + (2.0 * rho_next / delta) * rc[i];   // line 10
    rho = rho_next;
  }
}

// Lanczos: m steps from the start vector v0 (normalised here), no reorthogonalisation;
// alpha[0..m-1], beta[0..m-1] define the tridiagonal T (beta[j] couples j and j+1; beta[m-1] is the
// residual norm).  fp64 (the paper runs this in fp32 on the GPU; the estimates only steer the
// preconditioner).  Returns the number of steps done (stops early on an invariant subspace).
int oracle_lanczos(int64_t n, const int64_t* rowptr, const int32_t* col, const double* val, const double* v0,
                   int m, double* alpha, double* beta) {
  std::vector<double> v(n), vp(n, 0.0), w(n);
  const double nrm = std::sqrt(dot(n, v0, v0));
  for (int64_t i = 0; i < n; ++i) v[i] = v0[i] / nrm;
  double bprev = 0.0;
  for (int j = 0; j < m; ++j) {
    spmv(n, rowptr, col, val, v.data(), w.data());
    for (int64_t i = 0; i < n; ++i) w[i] -= bprev * vp[i];
    const double a = dot(n, w.data(), v.data());
    for (int64_t i = 0; i < n; ++i) w[i] -= a * v[i];
    const double bj = std::sqrt(dot(n, w.data(), w.data()));
    alpha[j] = a;
    beta[j] = bj;
    if (!(bj > 0.0)) return j + 1;
    for (int64_t i = 0; i < n; ++i) { vp[i] = v[i]; v[i] = w[i] / bj; }
    bprev = bj;
  }
  return m;
}

// Alg. 1 with M^-1 = Alg. 3.  Same stopping rule as oracle_pcg (R-G7).
int oracle_pcg_cheb(int64_t n, const int64_t* rowptr, const int32_t* col, const double* val, const double* b,
                    double* x, double rtol, int64_t max_iters, double lmin, double lmax, int k,
                    int64_t* iters_out, double* relres_true_out) {
  std::vector<double> r(n), z(n), p(n), mu(n);
  const double bnorm = std::sqrt(dot(n, b, b));
  int64_t it = 0;
  int status = 1;
  if (bnorm == 0.0) {
    std::memset(x, 0, sizeof(double) * n);
    *iters_out = 0; *relres_true_out = 0.0;
    return 0;
  }
  const double tol = rtol * bnorm;
  spmv(n, rowptr, col, val, x, mu.data());
  for (int64_t i = 0; i < n; ++i) r[i] = b[i] - mu[i];                         // line 1
  oracle_cheb_apply(n, rowptr, col, val, r.data(), lmin, lmax, k, z.data());   // line 2
  p = z;                                                                       // line 3
  double rho = dot(n, r.data(), z.data());
  double rnorm = std::sqrt(dot(n, r.data(), r.data()));
  double rel_true = rnorm / bnorm;
  for (;;) {
    if (rnorm <= tol) {
      spmv(n, rowptr, col, val, x, mu.data());
      for (int64_t i = 0; i < n; ++i) mu[i] = b[i] - mu[i];
      const double tn = std::sqrt(dot(n, mu.data(), mu.data()));
      rel_true = tn / bnorm;
      if (tn <= tol) { status = 0; break; }
      r = mu;
      oracle_cheb_apply(n, rowptr, col, val, r.data(), lmin, lmax, k, z.data());
      p = z;
      rho = dot(n, r.data(), z.data());
      rnorm = tn;
    }
    if (it >= max_iters) { status = 1; break; }
    spmv(n, rowptr, col, val, p.data(), mu.data());                            // line 6
    const double pmu = dot(n, p.data(), mu.data());
    if (!(pmu > 0.0) || !std::isfinite(pmu) || !std::isfinite(rho)) { status = 2; break; }
    const double alpha = rho / pmu;                                            // line 7
    for (int64_t i = 0; i < n; ++i) { x[i] += alpha * p[i]; r[i] -= alpha * mu[i]; }   // lines 8-9
    oracle_cheb_apply(n, rowptr, col, val, r.data(), lmin, lmax, k, z.data()); // line 10
    const double rho_new = dot(n, r.data(), z.data());
    const double beta = rho_new / rho;                                         // line 11
    for (int64_t i = 0; i < n; ++i) p[i] = z[i] + beta * p[i];                 // line 12
    rho = rho_new;
    rnorm = std::sqrt(dot(n, r.data(), r.data()));
    ++it;
  }
  if (status != 0) {
    spmv(n, rowptr, col, val, x, mu.data());
    for (int64_t i = 0; i < n; ++i) mu[i] = b[i] - mu[i];
    rel_true = std::sqrt(dot(n, mu.data(), mu.data())) / bnorm;
  }
  *iters_out = it;
  *relres_true_out = rel_true;
  return status;
}

}  // extern "C"
